#!/usr/bin/env python
"""Benchmark of the batched Generals.io environment step (BASELINE.json metric: 1v1 env steps/s on one B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch: gen_step for all N games (sampler -> moves /
combat / capture -> growth -> scoreboard / reward / done / auto-reset -> fog-of-war planes for both
players written to HBM).  value = env steps/s = games advanced one turn per second, whole job.
Workload: BASELINE config 2 (1v1 24x24, 16,384 games, auto-reset, four planes per player every step),
synthetic seeded boards.  One JSON line on stdout (rank 0).

--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same
workload: a deliberately plain program, reported as a baseline only.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "env steps/sec (1v1, all games) on 1 B200; % of HBM or int-issue roofline"
UNIT = "env_steps/s"
WORKLOAD = "c2_24x24"
HBM_FALLBACK_GBS = 6650.0          # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# dram bytes of one k_features launch (ncu --set full), by games per launch; see profiles/r01_features_full_summary.txt
NCU_FEAT_DRAM_BYTES_PER_LAUNCH = {16384: 3601662088}  # profiles/r01_features_full_summary.txt (k_features)


def algorithmic_bytes_per_env_step(H, W, P, packed=False):
    """SURVEY 8(d) B_min: read state 4*HW, write observations 5*P*HW (3*P*HW in the packed format, R33),
    O(P) scalars (actions 4P, reward P, done + winner 2, scoreboard 8P, turn 4)."""
    return 4 * H * W + (3 if packed else 5) * P * H * W + 13 * P + 6


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    return HBM_FALLBACK_GBS, "B200_PROFILING.md fallback (of fallback)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ reference arm
def oracle_throughput(cfg, sample_games, steps, warmup):
    """The oracle as it stands, single-threaded, on the first `sample_games` global game ids."""
    from oracle import oracle
    o = oracle.Oracle(dict(cfg, n_games=sample_games))
    o.reset()
    for _ in range(warmup):
        o.step()
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step()
    dt = time.perf_counter() - t0
    return sample_games * steps / dt, dt


def _oracle_worker(job):
    cfg, base, games, steps = job
    v, dt = oracle_throughput(dict(cfg, game_id_base=base), games, steps, 3)
    return games * steps, dt


def oracle_throughput_all_cores(cfg, games_per_core, steps):
    """one oracle process per host core over disjoint game-id ranges (the oracle itself stays
    single-threaded); aggregate env steps/s = all steps / the slowest process's time."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    jobs = [(cfg, c * games_per_core, games_per_core, steps) for c in range(cores)]
    with mp.get_context("spawn").Pool(cores) as pool:
        out = pool.map(_oracle_worker, jobs)
    return sum(n for n, _ in out) / max(dt for _, dt in out), cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import workloads
    cfg, _ = workloads.config(WORKLOAD)
    sample = 1024                      # config 2's first 1,024 games
    steps = min(args.steps, 500)
    value, dt = oracle_throughput(cfg, sample, steps, min(args.warmup, 20))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": min(args.warmup, 20), "ms_per_step": 1e3 * dt / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int16", "data": "synthetic",
        "config": {"workload": f"{WORKLOAD}: 1v1 24x24, auto-reset, sampler policy 5% pass; each step = "
                               f"first {sample} of 16,384 games advanced one turn by the CPU oracle"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"first {sample} global game ids x {steps} turns, single thread"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0



# ------------------------------------------------------------------------------------------ parity of the timed legs
PARITY_STATE = ["army", "owner", "terrain", "turn", "episode", "alive", "general_cell", "land", "army_total",
                "episodes_done", "wins", "truncations", "sat_events"]
PARITY_OUT = ["reward", "done", "winner", "obs_army", "obs_owner", "obs_terrain", "obs_vis"]


def parity_check(envs, mode="step", K=1, n_ids=8, actions=None, host_results=None):
    """after a timed leg and OUTSIDE every timed region, the CPU oracle (oracle/, the same test
    infrastructure the cpu_baseline leg times) replays `n_ids` games of the environments that leg stepped -- first, last
    and strided ids, split over `envs` -- for all the turns each environment has played since its last reset, through
    the same call sequence (mode "step": gen_step with the sampler; "rollout": gen_rollout(K, DIGEST); "every":
    gen_rollout(K, EVERY_STEP), all K slots compared; "actions": gen_step with the explicit action stream `actions`
    [T][N][P]).  Every state tensor, the scoreboard, reward / done / winner and the four observation planes of those
    games (plus the chained digest in mode "rollout", plus the host copies `host_results` = (reward, done) of the last
    step in mode "actions") must be bit-equal.  Returns the JSON object {"games", "turns", "ok", ...}."""
    import numpy as np
    import torch
    from oracle import oracle
    per_env = max(1, n_ids // len(envs))
    games, turns, bad = 0, 0, None
    for env in envs:
        torch.cuda.synchronize()
        N, T = env.N, env.global_step
        ids = sorted({(k * (N - 1)) // max(1, per_env - 1) for k in range(per_env)})
        sel = torch.tensor(ids, device=env.device)
        slots = K if mode == "every" else 1
        fields = PARITY_STATE + PARITY_OUT + (["obs_digest"] if mode == "rollout" else [])
        got = [{f: (env.tensors[f][k] if f in PARITY_OUT else env.tensors[f]).index_select(0, sel).cpu().numpy()
                for f in fields if k == 0 or f in PARITY_OUT} for k in range(slots)]
        for j, g in enumerate(ids):
            cfg1 = dict(env.cfg_dict, n_games=1, game_id_base=env.cfg_dict.get("game_id_base", 0) + g)
            o = oracle.Oracle(cfg1, every_step_K=K if mode == "every" else 0, digest=(mode == "rollout"))
            o.reset()
            if mode == "step":
                for _ in range(T):
                    o.step()
            elif mode == "actions":
                for t in range(T):
                    o.step(actions[t, g].numpy().reshape(1, -1))
            else:
                for _ in range(T // K):
                    o.rollout(K, oracle.OBS_EVERY_STEP if mode == "every" else oracle.OBS_DIGEST)
            for k in range(slots):
                for f, have in got[k].items():
                    want = np.asarray(getattr(o, f))
                    want = want[k][0] if f in PARITY_OUT else want[0]
                    if have[j].dtype != want.dtype:
                        want = want.view(have[j].dtype) if want.ndim else np.asarray(want).astype(have[j].dtype)
                    if not np.array_equal(have[j], want.reshape(have[j].shape)) and bad is None:
                        bad = {"game": int(cfg1["game_id_base"]), "field": f, "slot": k}
            if host_results is not None and bad is None:
                hr, hd = host_results
                if not (np.array_equal(hr.numpy()[g], o.reward[0][0]) and int(hd.numpy()[g]) == int(o.done[0][0])):
                    bad = {"game": int(cfg1["game_id_base"]), "field": "host reward / done"}
        games += len(ids)
        turns = max(turns, T)
    out = {"games": games, "turns": turns, "ok": bad is None, "against": "oracle/ replay of the sampled games, all "
           "state tensors, scoreboard, reward / done / winner and observation planes bit-equal"}
    if bad is not None:
        out["first_mismatch"] = bad
    return out


# ------------------------------------------------------------------------------------------ our arm
MIN_REGION_MS, MIN_REPS, MAX_REPS = 50.0, 5, 60
PHASE_STRIDE = 160                  # turns between the starting phases of consecutive replicas of the headline rotation
# warp-instructions per env step of the fused rollout kernel (gen_rollout(32, GEN_OBS_DIGEST), 24x24 1v1):
# smsp__inst_executed.sum / (N * K) of the ncu capture summarised in the file named beside it
ROLLOUT_INST_PER_ENV_STEP = 659.4
ROLLOUT_INST_SOURCE = "profiles/r02_rollout_summary.txt"
# the method's own work per env step as SURVEY 8(d) estimates it ("3-4 x 10^2 warp-instructions" at 24x24 1v1: fog test +
# selects + mix per visible cell and player, growth, sampler, moves); the kernel executes more than that (index
# arithmetic, staging, reductions), so frac_algorithmic < frac says how much of the issued work is overhead
ROLLOUT_ALGORITHMIC_INST_PER_ENV_STEP = 350.0
ISSUE_PEAK = 148 * 4 * 1.965e9      # warp-instructions/s: 148 SMs x 4 schedulers x 1 per clock x 1.965 GHz
# dram__bytes_read.sum + dram__bytes_write.sum per launch of k_step at N = 262,144 (ncu --set full), by games per launch
NCU_DRAM_BYTES_PER_LAUNCH_LARGE = {262144: (2303562752, "profiles/r02_step_full_262k_summary.txt")}
# the same for the headline rotation (six replicas of 16,384 games, caches left alone between launches: mean of 36
# consecutive launches, ncu --cache-control none)
NCU_DRAM_BYTES_PER_LAUNCH = {16384: (144697216, "profiles/r03_rotation_dram.md")}


def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads
    from paper_2606_23348_b200 import GeneralsEnv, OBS_DIGEST, OBS_EVERY_STEP, OBS_NONE, replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg, _ = workloads.config(WORKLOAD)
    if args.games:
        cfg["n_games"] = args.games
    N, P, H, W = cfg["n_games"], cfg["n_players"], cfg["height"], cfg["width"]
    bmin = algorithmic_bytes_per_env_step(H, W, P)
    K, Wm = args.steps, args.warmup
    peak, peak_src = measured_peak()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return replicas.max_over_ranks(x, dist if world > 1 else None, dev)

    def event():
        return torch.cuda.Event(enable_timing=True)

    def timed(launch_k, k):
        """Repetitions of exactly k calls of launch_k's body under one CUDA event pair each (barrier + synchronize on
        both sides, max over ranks), repeated at least MIN_REPS times and until the repetitions add up to
        MIN_REGION_MS: SURVEY 8(d) 'best and median of 5'.  Returns the list of ms per repetition."""
        reps = []
        while len(reps) < MIN_REPS or (sum(reps) < MIN_REGION_MS and len(reps) < MAX_REPS):
            e0, e1 = event(), event()
            barrier()
            e0.record()
            launch_k(k)
            e1.record()
            barrier()
            reps.append(max_over_ranks(e0.elapsed_time(e1)))
        return reps

    def summary(reps, k, n_games):
        med, best = statistics.median(reps), min(reps)
        return {"value": world * n_games * k / (med * 1e-3), "best": world * n_games * k / (best * 1e-3), "unit": UNIT,
                "us_per_launch": 1e3 * med / k, "best_us_per_launch": 1e3 * best / k, "repetitions": len(reps),
                "launches_per_repetition": k}

    def checked(envs_, **kw):
        # the oracle is test infrastructure: it runs here only beside the cpu_baseline leg, never inside a timed region
        return None if args.no_cpu_baseline else parity_check(envs_, **kw)

    def make_replicas(cfg_r, n_games, count, actions_out_first=False):
        out = []
        for r in range(count):
            c = replicas.weak_replica_config(dict(cfg_r, n_games=n_games, game_id_base=0), rank * count + r)
            out.append(GeneralsEnv(c, device=dev, digest=False, actions_out=(actions_out_first and r == 0)))
            out[-1].cfg_dict = c
        return out

    # Replicas of the batch, stepped round-robin, so that every launch finds its inputs in HBM and not in
    # the 126 MB L2: between two steps of the same replica the others move (R - 1) * N * bmin bytes.
    R = args.replicas or max(2, -(-(640 << 20) // (N * bmin)))
    envs = make_replicas(cfg, N, R, actions_out_first=True)
    env = envs[0]

    # ---- record the action stream of warm-up + timed steps for the end-to-end leg (device sampler -> host)
    env.reset()
    h_actions = torch.empty((Wm + K, N, P), dtype=torch.int32).pin_memory()
    for t in range(Wm + K):
        env.step()
        h_actions[t].copy_(env.tensors["actions_out"][0], non_blocking=True)
    torch.cuda.synchronize()

    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()                                       # sampling spans warm-up and every timed leg below

    # ---- headline: K gen_step launches back to back, replica t % R at step t
    # Phase mix: an episode of config 2 runs 1,000 turns and the board fills up on the way, so replica
    # r is first played forward to turn r * PHASE_STRIDE with one state-only fused rollout (untimed); the timed launches
    # then sample early, middle and late game and, on the last replica, the truncation + auto-reset at turn 1,000.
    for r, e in enumerate(envs):
        e.reset()
        if r and not args.no_phase_mix:
            e.rollout(r * PHASE_STRIDE, OBS_NONE)
    for t in range(max(Wm, 2 * R)):                          # every replica stepped at least twice before timing
        envs[t % R].step()
    torch.cuda.synchronize()
    turns_before = [e.global_step for e in envs]
    counter = [0]

    def rotate(k):
        t0 = counter[0]
        for t in range(t0, t0 + k):
            envs[t % R].step()
        counter[0] = t0 + k

    launches0 = sum(e.launch_count for e in envs)
    reps = timed(rotate, K)
    launches = (sum(e.launch_count for e in envs) - launches0) // len(reps)
    head = summary(reps, K, N)
    total_ms = statistics.median(reps)
    head_parity = checked([envs[0], envs[R - 1]])
    turns_timed = [f"{a}-{e.global_step}" for a, e in zip(turns_before, envs)]
    specialised, reg_resident = env.last_launch_specialised, env.last_launch_register_resident

    # ---- one environment stepped K times back to back (launch t+1 depends on launch t game by game; the 132 MB
    # working set of one batch is partly L2-resident, so this is NOT the roofline leg)
    def same(k):
        for _ in range(k):
            env.step()

    same(Wm)
    same_env = summary(timed(same, K), K, N)
    same_parity = checked([env])

    # ---- isolated launches: a 256 MB L2-flush write before every launch and one event pair per launch (includes
    # the launch latency a back-to-back stream hides); what a loop with other kernels between the steps gets
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = [(event(), event()) for _ in range(60)]
    barrier()
    for a, b in ev:
        flush.fill_(1)
        a.record()
        env.step()
        b.record()
    barrier()
    iso = sorted(a.elapsed_time(b) for a, b in ev)
    iso_med, iso_best = max_over_ranks(statistics.median(iso)), max_over_ranks(iso[0])
    del flush

    # ---- interleaved: a foreign kernel of about 10 us (the policy stand-in: a 24 MB fill) between two steps of ONE
    # environment -- launches cannot chain across it; cost of a step = pair - foreign alone
    foreign = torch.empty(24 << 20, dtype=torch.uint8, device=dev)

    def only_foreign(k):
        for _ in range(k):
            foreign.fill_(3)

    def pair(k):
        for _ in range(k):
            foreign.fill_(3)
            env.step()

    pair(Wm)
    f_reps, p_reps = timed(only_foreign, K), timed(pair, K)
    f_us, p_us = 1e3 * statistics.median(f_reps) / K, 1e3 * statistics.median(p_reps) / K
    inter_parity = checked([env])                            # covers the isolated launches before it as well
    # the same with TWO environments on two streams (the usual schedule of a learner with two env batches: the policy
    # works on one while the other steps): each stream alternates its foreign kernel and its step
    side = [torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)]
    foreign2 = torch.empty(24 << 20, dtype=torch.uint8, device=dev)
    two_envs, two_bufs = [envs[0], envs[1]], [foreign, foreign2]

    def on_two_streams(body):
        def run(k):
            cur = torch.cuda.current_stream(dev)
            for st in side:
                st.wait_stream(cur)
            for _ in range(k):
                for i in range(2):
                    with torch.cuda.stream(side[i]):
                        body(i)
            for st in side:
                cur.wait_stream(st)
        return run

    def two_pair(i):
        two_bufs[i].fill_(3)
        two_envs[i].step(stream=side[i])

    on_two_streams(two_pair)(Wm)
    f2_reps = timed(on_two_streams(lambda i: two_bufs[i].fill_(3)), K)
    p2_reps = timed(on_two_streams(two_pair), K)
    f2_us, p2_us = 1e3 * statistics.median(f2_reps) / (2 * K), 1e3 * statistics.median(p2_reps) / (2 * K)
    two_parity = checked(two_envs)
    del foreign, foreign2, two_bufs

    # ---- gen_step + gen_features (bfloat16 feature tensor, R37) every turn: the featuriser between two steps
    fenv = envs[1]
    fenv.reset()
    fenv.features(bf16=True)

    def only_features(k):
        for _ in range(k):
            fenv.features()

    def step_features(k):
        for _ in range(k):
            fenv.step()
            fenv.features()

    step_features(max(Wm, 8))
    sf_reps = timed(step_features, max(8, K // 4))
    of_reps = timed(only_features, max(8, K // 4))     # same turn folded again: same traffic, memory unchanged
    sf_us, of_us = 1e3 * statistics.median(sf_reps) / max(8, K // 4), 1e3 * statistics.median(of_reps) / max(8, K // 4)
    del fenv.feat_tensors, fenv.feat
    del fenv.feat_bufs

    # ---- fused rollout leg (K_r = 32 turns per launch, observation digest chained every turn)
    renv = GeneralsEnv(replicas.weak_replica_config(cfg, rank), device=dev, digest=True, actions_out=False)
    renv.cfg_dict = replicas.weak_replica_config(cfg, rank)
    renv.reset()
    renv.rollout(32, OBS_DIGEST)
    n_roll = max(2, K // 32)

    def roll(k):
        for _ in range(k):
            renv.rollout(32, OBS_DIGEST)

    roll_reps = timed(roll, n_roll)
    roll_value = world * N * 32 * n_roll / (statistics.median(roll_reps) * 1e-3)
    roll_parity = checked([renv], mode="rollout", K=32)
    roll_variant = renv.lib.gen_last_variant(renv._env, None, None)
    del renv
    # ---- fused rollout with the planes of EVERY turn written (K = 8 slots): the same output as eight gen_step
    # launches with the built-in sampler, the state read once per launch
    KE = 8
    eenv = GeneralsEnv(replicas.weak_replica_config(cfg, rank), device=dev, k_slots=KE, digest=False, actions_out=False)
    eenv.cfg_dict = replicas.weak_replica_config(cfg, rank)
    eenv.reset()
    eenv.rollout(KE, OBS_EVERY_STEP)
    n_every = max(2, K // KE)

    def roll_every(k):
        for _ in range(k):
            eenv.rollout(KE, OBS_EVERY_STEP)

    every_reps = timed(roll_every, n_every)
    every_value = world * N * KE * n_every / (statistics.median(every_reps) * 1e-3)
    every_bytes = bmin - 4 * H * W * (KE - 1) / KE
    every_parity = checked([eenv], mode="every", K=KE)
    every_variant = eenv.lib.gen_last_variant(eenv._env, None, None)
    del eenv

    # ---- end-to-end leg: host actions in (pinned), gen_step_host, host reward + done out, every step
    env.reset()
    h_reward = torch.zeros((N, P), dtype=torch.int8).pin_memory()
    h_done = torch.zeros((N,), dtype=torch.uint8).pin_memory()
    for t in range(Wm):
        env.step_host(h_actions[t], h_reward, h_done)
    e2e_reps = []
    for _ in range(MIN_REPS):
        env.reset()
        for t in range(Wm):
            env.step_host(h_actions[t], h_reward, h_done)
        barrier()
        t0 = time.perf_counter()
        for t in range(Wm, Wm + K):
            env.step_host(h_actions[t], h_reward, h_done)
        torch.cuda.synchronize()
        e2e_reps.append(max_over_ranks(time.perf_counter() - t0))
    e2e_s = statistics.median(e2e_reps)
    # the same loop without a synchronisation per step: gen_step_host_async, two sets of pinned result slots, the
    # results of step t - 1 read (gen_host_wait(1)) after step t has been issued
    slots = [(torch.zeros((N, P), dtype=torch.int8).pin_memory(), torch.zeros((N,), dtype=torch.uint8).pin_memory())
             for _ in range(2)]
    async_reps, async_sum = [], 0                            # async_sum: the host really reads a result every step
    for _ in range(MIN_REPS):
        env.reset()
        for t in range(Wm):
            env.step_host(h_actions[t], h_reward, h_done)
        barrier()
        t0 = time.perf_counter()
        for t in range(Wm, Wm + K):
            r, d = slots[t & 1]
            env.step_host_async(h_actions[t], r, d)
            if t > Wm:
                env.host_wait(1)
                async_sum += int(slots[(t - 1) & 1][1][0])       # the host reads a result of step t - 1
        env.host_wait(0)
        async_sum += int(slots[(Wm + K - 1) & 1][1][0])
        async_reps.append(max_over_ranks(time.perf_counter() - t0))
    async_s = statistics.median(async_reps)
    e2e_parity = checked([env], mode="actions", actions=h_actions, host_results=slots[(Wm + K - 1) & 1])
    e2e_variant = env.lib.gen_last_variant(env._env, None, None)

    # ---- large batch ("quote the fraction from N >= 262,144"): the same kernel where one launch is
    # 22 waves and the batch (2.1 GB of state + observations per replica) is far larger than L2
    large = None
    if not args.no_large and not args.games:
        del envs, env, fenv
        torch.cuda.empty_cache()
        NL = 262144
        lenvs = make_replicas(cfg, NL, 2)
        for e in lenvs:
            e.reset()
        lc = [0]

        def lrot(k):
            for t in range(lc[0], lc[0] + k):
                lenvs[t % 2].step()
            lc[0] += k

        lrot(6)
        KL = max(8, min(K, 20))
        l_reps = timed(lrot, KL)
        large = summary(l_reps, KL, NL)
        large["parity_checked"] = checked(lenvs)
        del lenvs
        torch.cuda.empty_cache()
        leenv = GeneralsEnv(replicas.weak_replica_config(dict(cfg, n_games=NL), rank), device=dev, k_slots=KE, digest=False,
                            actions_out=False)
        leenv.cfg_dict = replicas.weak_replica_config(dict(cfg, n_games=NL), rank)
        leenv.reset()
        leenv.rollout(KE, OBS_EVERY_STEP)

        def lroll_every(k):
            for _ in range(k):
                leenv.rollout(KE, OBS_EVERY_STEP)

        le_reps = timed(lroll_every, 4)
        large["rollout_every_step"] = world * NL * KE * 4 / (statistics.median(le_reps) * 1e-3)
        large["rollout_every_parity"] = checked([leenv], mode="every", K=KE)
        del leenv
        torch.cuda.empty_cache()

    # The timed regions above last tens of milliseconds each, nvidia-smi samples every 100 ms: the sampler has seen the
    # GPU under this load several times by now.
    clock_info = clocks.stop() if rank == 0 else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    launch_ms = total_ms / K
    achieved = N * bmin / (launch_ms * 1e-3) / 1e9
    kname = ("gen::k_step" if reg_resident else "gen::k_generals") + (f"<{P}, {H}, {W}>" if specialised else " (generic)")
    iso_ach = N * bmin / (iso_med * 1e-3) / 1e9
    step_us_inter = p_us - f_us
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int16", "data": "synthetic",
        "config": {"workload": f"{WORKLOAD}: 1v1 24x24, {N} games/GPU, auto-reset, max_turns 1000, device Philox "
                               "sampler 5% pass, 4 obs planes x 2 players written every step",
                   "n_games_per_gpu": N, "path": "gen_step (per-step kernel, 1 launch per step)",
                   "l2": f"inputs larger than L2: {R} replicas of the batch stepped round-robin ({R} x "
                         f"{N * bmin / 1e6:.0f} MB of algorithmic traffic between two steps of one replica; L2 is "
                         "126 MB); K launches back to back, one CUDA event pair around them",
                   "replicas_in_rotation": R,
                   "turns_timed": "turns of the episode each replica played inside the timed repetitions (replica r "
                                  f"pre-rolled to turn r x {PHASE_STRIDE}; max_turns 1000): " + ", ".join(turns_timed),
                   "timing": f"value = median of {len(reps)} repetitions of exactly {K} launches (one event pair each, "
                             f"barrier + synchronize on both sides; repeated until >= {MIN_REGION_MS:.0f} ms in total); "
                             "best repetition in value_best",
                   "parallelism": f"replicas x{world}, disjoint game-id ranges, no collective"},
        "value_best": head["best"], "repetitions": len(reps),
        "parity_checked": head_parity,
        "clocks": clock_info,
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": (NCU_DRAM_BYTES_PER_LAUNCH.get(N) or (None, None))[0],
                     "traffic_source": (NCU_DRAM_BYTES_PER_LAUNCH.get(N) or (None, None))[1],
                     "traffic_over_algorithmic": (NCU_DRAM_BYTES_PER_LAUNCH[N][0] / (N * bmin)
                                                  if N in NCU_DRAM_BYTES_PER_LAUNCH else None),
                     "kernel": kname + " (gen_step)", "peak_source": peak_src,
                     "algorithmic_bytes_per_env_step": bmin, "units_per_launch": N,
                     "avg_launch_us": 1e3 * launch_ms, "best_launch_us": head["best_us_per_launch"],
                     "isolated_launch_us": 1e3 * iso_med},
        "roofline_isolated": {"bound": "hbm", "achieved": iso_ach, "peak": peak, "unit": "GB/s", "frac": iso_ach / peak,
                              "launch_us": 1e3 * iso_med, "best_launch_us": 1e3 * iso_best, "launches": len(iso),
                              "note": "median of single launches, each after a 256 MB L2-flush write and with its own "
                                      "event pair (launch latency included): one gen_step by itself, nothing to overlap with"},
        "interleaved": {"value": world * N / (step_us_inter * 1e-6), "unit": UNIT, "pair_us": p_us, "foreign_us": f_us,
                        "step_us": step_us_inter, "frac": N * bmin / (step_us_inter * 1e-6) / 1e9 / peak,
                        "repetitions": len(p_reps),
                        "note": "one environment; a foreign kernel (24 MB fill, the policy stand-in) between two steps, "
                                "so launches cannot chain; step_us = pair - foreign alone",
                        "parity_checked": inter_parity},
        "interleaved_two_batches": {"loop_value": world * N / (p2_us * 1e-6), "loop_value_one_batch": world * N / (p_us * 1e-6),
                                    "unit": UNIT, "pair_us": p2_us, "foreign_us": f2_us, "step_us": p2_us - f2_us,
                                    "repetitions": len(p2_reps),
                                    "note": "two environments on two streams, each alternating a foreign kernel (24 MB fill) "
                                            "and its step -- the schedule of a learner with two env batches: one batch's store "
                                            "phase runs under the other's foreign kernel and rules.  loop_value = env steps/s of "
                                            "the whole loop, foreign kernels included (one batch on one stream beside it); "
                                            "pair_us = time per (foreign + step) pair; step_us = pair - foreign alone attributes "
                                            "ALL of the overlap to the step and is not a roofline figure",
                                    "parity_checked": two_parity},
        "step_plus_features": {"turn_us": sf_us, "features_us": of_us, "step_us": sf_us - of_us,
                               "value": world * N / (sf_us * 1e-6), "unit": UNIT, "dtype": "bf16 feature tensor (R37)",
                               "note": "gen_step + gen_features every turn (38 channels x 2 players materialised)"},
        "e2e": {"value": world * N * K / async_s, "unit": UNIT, "h2d_bytes_per_step": N * P * 4,
                "d2h_bytes_per_step": N * P + N,
                "best": world * N * K / min(async_reps), "repetitions": len(async_reps),
                "api": "gen_step_host_async + gen_host_wait(1): pinned host actions read in place, reward + done written "
                       "by the step kernel into two alternating sets of pinned host arrays, the host reads the results of "
                       "step t - 1 after issuing step t (no synchronisation per step, no second kernel); the observation planes stay on the device BY "
                       "DESIGN (a GPU-resident learner reads them there: 94 MB per step is no bus traffic to plan for) "
                       "and are not part of the returned result",
                "synchronised_every_step": {"value": world * N * K / e2e_s, "best": world * N * K / min(e2e_reps),
                                            "api": "gen_step_host (cudaStreamSynchronize per step)"},
                "parity_checked": e2e_parity, "kernel_variant": e2e_variant},
        "same_env": dict(same_env, parity_checked=same_parity, note="one environment stepped K times back to back (true game-by-game dependency "
                                        "between launches; working set partly L2-resident: not a roofline figure)"),
        "rollout": {"value": roll_value, "unit": UNIT, "K": 32, "launches": n_roll, "repetitions": len(roll_reps),
                    "obs": "digest every turn, planes of the last turn",
                    "parity_checked": roll_parity, "kernel_variant": roll_variant,
                    "roofline": {"bound": "alu", "inst_per_env_step": ROLLOUT_INST_PER_ENV_STEP,
                                 "inst_source": ROLLOUT_INST_SOURCE,
                                 "achieved": roll_value / world * ROLLOUT_INST_PER_ENV_STEP, "peak": ISSUE_PEAK,
                                 "unit": "warp-inst/s", "frac": roll_value / world * ROLLOUT_INST_PER_ENV_STEP / ISSUE_PEAK,
                                 "algorithmic_inst_per_env_step": ROLLOUT_ALGORITHMIC_INST_PER_ENV_STEP,
                                 "algorithmic_source": "SURVEY.md 8(d) estimate (3-4e2 warp-instructions per env step)",
                                 "frac_algorithmic": roll_value / world * ROLLOUT_ALGORITHMIC_INST_PER_ENV_STEP / ISSUE_PEAK}},
        "rollout_every_step": {"value": every_value, "unit": UNIT, "K": KE, "launches": n_every, "repetitions": len(every_reps),
                               "parity_checked": every_parity, "kernel_variant": every_variant,
                               "obs": "four planes x 2 players of EVERY turn, K-strided slots (what K gen_step launches with "
                                      "the built-in sampler write)",
                               "roofline": {"bound": "hbm", "algorithmic_bytes_per_env_step": every_bytes,
                                            "achieved": every_value / world * every_bytes / 1e9, "peak": peak, "unit": "GB/s",
                                            "frac": every_value / world * every_bytes / 1e9 / peak,
                                            "kernel": "gen::k_generals<2, 24, 24, F_OBS_PLANES | F_OBS_EVERY> (gen_rollout)"}},
    }
    if large:
        NL = 262144
        l_ach = NL * bmin / (large["us_per_launch"] * 1e-6) / 1e9
        tr = NCU_DRAM_BYTES_PER_LAUNCH_LARGE.get(NL)
        line["roofline_large"] = {"bound": "hbm", "achieved": l_ach, "peak": peak, "unit": "GB/s", "frac": l_ach / peak,
                                  "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None,
                                  "traffic_over_algorithmic": tr[0] / (NL * bmin) if tr else None,
                                  "value": large["value"], "best": large["best"], "units_per_launch": NL,
                                  "parity_checked": large["parity_checked"],
                                  "avg_launch_us": large["us_per_launch"], "repetitions": large["repetitions"],
                                  "launches_per_repetition": large["launches_per_repetition"],
                                  "kernel": kname + " (gen_step), 2 replicas of 262,144 games in rotation",
                                  "rollout_every_step": {"value": large["rollout_every_step"], "unit": UNIT, "K": KE,
                                                         "frac": large["rollout_every_step"] / world * every_bytes / 1e9 / peak,
                                                         "parity_checked": large["rollout_every_parity"],
                                                         "note": "gen_rollout(8, GEN_OBS_EVERY_STEP) at the same batch size"}}
    if not args.no_cpu_baseline:
        # config 2's first 1,024 games; 500 turns instead of 2,000 so that the leg stays near 20 s of CPU
        sample, steps = 1024, 500
        v, _ = oracle_throughput(dict(cfg, game_id_base=0), sample, steps, 5)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"first {sample} global game ids x {steps} turns of {WORKLOAD}, single thread "
                                          "(SURVEY 8(d) names 2,000 turns: bounded to about 20 s of CPU work)"}
        c1, t1 = workloads.config("c1_8x8")
        v1, _ = oracle_throughput(c1, c1["n_games"], t1, 0)
        line["cpu_baseline_config1"] = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle",
                                        "sample": "config 1 in full: 64 games x 300 turns, 8x8, single thread"}
        try:
            va, cores = oracle_throughput_all_cores(dict(cfg), 64, 300)
            line["cpu_baseline_all_cores"] = {"value": va, "unit": UNIT, "cores": cores, "kind": "oracle",
                                              "sample": f"one single-threaded oracle process per host core, 64 games x "
                                                        f"300 turns of {WORKLOAD} each, disjoint global game ids"}
        except Exception as exc:                                   # a baseline, never a reason to lose the line
            line["cpu_baseline_all_cores"] = {"value": None, "error": repr(exc)}
    for k in ("same_env", "interleaved_two_batches", "interleaved", "roofline_isolated"):
        line[k] = line.pop(k)             # last in the line: a log that keeps only the tail of stdout keeps these
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_single_leg(args):
    """--only rollout | step | step-large: one leg by itself, a handful of launches -- the command the ncu captures under
    profiles/ are taken with (ncu replays every kernel it profiles ~40 times: a full bench run under it takes long)."""
    import torch
    import workloads
    from paper_2606_23348_b200 import GeneralsEnv, OBS_DIGEST
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    n = {"rollout": 16384, "step": 16384, "step-large": 262144, "rotation": 16384, "noalloc": 16384}[args.only]
    cfg, _ = workloads.config(args.workload or WORKLOAD, n_games=args.games or n)
    if args.only == "rotation":
        # the headline leg by itself: R replicas of the batch (640 MB of algorithmic traffic between two steps of one
        # replica), pre-rolled to different phases of the episode, stepped round-robin -- the command of the
        # dram__bytes capture behind roofline.traffic (ncu --cache-control none: the caches carry over from launch to
        # launch as they do in the timed run)
        from paper_2606_23348_b200 import OBS_NONE
        N = cfg["n_games"]
        bmin = algorithmic_bytes_per_env_step(cfg["height"], cfg["width"], cfg["n_players"])
        R = args.replicas or max(2, -(-(640 << 20) // (N * bmin)))
        envs = [GeneralsEnv(dict(cfg, game_id_base=r * N), device=dev, digest=False, actions_out=False) for r in range(R)]
        for r, e in enumerate(envs):
            e.reset()
            if r and not args.no_phase_mix:
                e.rollout(r * PHASE_STRIDE, OBS_NONE)
        for t in range(2 * R):
            envs[t % R].step()
        k = max(2 * R, min(args.steps, 400))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for t in range(k):
            envs[t % R].step()
        e1.record()
        torch.cuda.synchronize()
        print(json.dumps({"leg": "rotation", "n_games": N, "replicas": R, "launches": k, "warmup_launches": 2 * R,
                          "us_per_launch": 1e3 * e0.elapsed_time(e1) / k,
                          "env_steps_per_s": N * k / (e0.elapsed_time(e1) * 1e-3),
                          "kernel_variant": envs[0].lib.gen_last_variant(envs[0]._env, None, None)}))
        return 0
    if args.only == "noalloc":
        # gen_step_noalloc (bitboard cache in the library's fixed device array, rebuilt per call, never chained) beside
        # gen_step with a caller-allocated cache on the same boards: what the convenience costs
        out = {"leg": "noalloc", "n_games": cfg["n_games"]}
        k = max(4, min(args.steps, 400))
        for name, kw in (("gen_step", {}), ("gen_step_noalloc", dict(bitboards=False, chain=False, stack_cache=False))):
            env = GeneralsEnv(cfg, device=dev, digest=False, actions_out=False, **kw)
            call = env.step_noalloc if kw else env.step
            env.reset()
            for _ in range(10):
                call()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            l0 = env.launch_count
            e0.record()
            for _ in range(k):
                call()
            e1.record()
            torch.cuda.synchronize()
            out[name] = {"us_per_call": 1e3 * e0.elapsed_time(e1) / k, "kernels_per_call": (env.launch_count - l0) / k,
                         "env_steps_per_s": cfg["n_games"] * k / (e0.elapsed_time(e1) * 1e-3)}
            del env
        out["note"] = "one environment stepped back to back (partly L2-resident: compare the two, not with the headline)"
        print(json.dumps(out))
        return 0
    env = GeneralsEnv(cfg, device=dev, digest=(args.only == "rollout"), actions_out=False)
    if args.force_step:
        env.set_generic(False, -1)      # the register-resident kernel also where the staged one is the default (P > 4)
    env.reset()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k = max(4, min(args.steps, 400))
    for _ in range(3):
        env.rollout(32, OBS_DIGEST) if args.only == "rollout" else env.step()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(k):
        env.rollout(32, OBS_DIGEST) if args.only == "rollout" else env.step()
    e1.record()
    torch.cuda.synchronize()
    turns = 32 if args.only == "rollout" else 1
    out = {"leg": args.only, "n_games": cfg["n_games"], "launches": k, "turns_per_launch": turns,
           "us_per_launch": 1e3 * e0.elapsed_time(e1) / k,
           "env_steps_per_s": cfg["n_games"] * turns * k / (e0.elapsed_time(e1) * 1e-3)}
    # Development builds (GEN_NVCC_FLAGS=-DGEN_TRACE python -m paper_2606_23348_b200.build --force) keep a per-warp
    # timeline of the per-step kernel (%globaltimer at every phase boundary): one lone launch after an L2 flush and
    # one behind a foreign kernel, summarised as mean / max time since the first warp started, in microseconds.
    variant = env.lib.gen_last_variant(env._env, None, None)
    reader = getattr(env.lib, f"gen_debug_trace_{variant}", None) if args.only == "step" else None
    if reader is not None:
        import ctypes
        import numpy as np
        names = ["start", "scalars", "rows", "sampler", "moves", "growth", "end_of_turn", "fog", "emit", "store"]
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        foreign = torch.empty(24 << 20, dtype=torch.uint8, device=dev)
        warps = min(8192, (cfg["n_games"] + 3) // 4)
        out["timeline_us"] = {}
        for tag, pre in (("lone_after_l2_flush", lambda: flush.fill_(1)), ("behind_foreign_kernel", lambda: foreign.fill_(3))):
            for _ in range(3):
                pre()
                torch.cuda.synchronize()
                env.step()
                torch.cuda.synchronize()
            buf = np.zeros(warps * 16, dtype=np.uint64)
            reader(buf.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(warps * 16))
            t = buf.reshape(warps, 16).astype(np.int64)
            t0 = t[:, 0].min()
            done = (t[:, 9] - t0) / 1e3
            out["timeline_us"][tag] = {
                "phase_end_mean_max": {n: [round(float((t[:, i].mean() - t0) / 1e3), 1), round(float((t[:, i].max() - t0) / 1e3), 1)]
                                       for i, n in enumerate(names)},
                "warps_finished_by_us": {str(b): int((done <= b).sum()) for b in (16, 20, 24, 28, 32, 36, 40)},
                "warps": warps}
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------------------------------ batch sweep
def time_steps(torch, envs, K, warm, graph):
    """K gen_step launches back to back, replica t % R at launch t; returns ms.  graph=True replays them as one
    CUDA graph (host launch cost out of the picture: what matters at small N)."""
    R = len(envs)
    for t in range(warm):
        envs[t % R].step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if graph:
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        with torch.cuda.graph(g, stream=side):
            for t in range(K):
                envs[t % R].step()
        torch.cuda.synchronize()
        e0.record()
        g.replay()
        e1.record()
    else:
        e0.record()
        for t in range(K):
            envs[t % R].step()
        e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def run_sweep(args):
    """BASELINE config 3 (batch sweep, per-step kernel vs fused K = 32 rollout) plus per-step rows for configs
    4 and 5: one JSON line per row.  Not the driver's contract line; its results are copied into BASELINE.md."""
    import torch
    import workloads
    from paper_2606_23348_b200 import GeneralsEnv, OBS_DIGEST
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = measured_peak()
    rows = [("c3_sweep", n, False) for n in (1024, 16384, 262144, 1048576)]
    rows += [("c4_curriculum", 65536, False), ("c5a_2v2", 32768, False), ("c5b_ffa8", 32768, False)]
    rows += [("c3_sweep", 16384, True), ("c3_sweep", 262144, True)]        # packed observation format (R33)
    rows += [("official_23x23", 16384, False), ("official_23x23", 262144, False)]   # official maps (R36, NEXT-3)
    for name, N, packed in rows:
        if args.rows and args.rows not in name:
            continue
        cfg, _ = workloads.config(name, n_games=N)
        P, H, W = cfg["n_players"], cfg["height"], cfg["width"]
        bmin = algorithmic_bytes_per_env_step(H, W, P, packed)
        R = max(2, -(-(640 << 20) // (N * bmin)))
        K = max(32, min(args.steps, (1 << 31) // (N * bmin) * 4))
        envs = [GeneralsEnv(dict(cfg, game_id_base=r * N), device=dev, digest=False, actions_out=False, packed=packed)
                for r in range(R)]
        for e in envs:
            e.reset()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        envs[0].reset()                                     # board generation for all N games + first observation
        e1.record()
        torch.cuda.synchronize()
        reset_ms = e0.elapsed_time(e1)
        out = {"workload": name, "reset_us": 1e3 * reset_ms, "maps_per_s": N / (reset_ms * 1e-3), "obs_format": "army + packed byte (R33)" if packed else "4 planes", "n_games": N, "n_players": P, "board": f"{H}x{W}", "replicas_in_rotation": R,
               "steps": K, "algorithmic_bytes_per_env_step": bmin}
        for graph in (False, True):
            ms = statistics.median(time_steps(torch, envs, K, max(args.warmup, R), graph) for _ in range(5))
            key = "step_graph" if graph else "step"
            out[key] = {"env_steps_per_s": N * K / (ms * 1e-3), "us_per_launch": 1e3 * ms / K,
                        "hbm_frac": N * bmin / (ms / K * 1e-3) / 1e9 / peak}
        out["kernel"] = ("k_step" if envs[0].last_launch_register_resident else "k_generals") + \
                        ("" if envs[0].last_launch_specialised else " (generic)")
        del envs
        torch.cuda.empty_cache()
        if name == "c3_sweep" and not packed and N <= 262144:
            # fused rollout with the planes of EVERY turn written to K-strided buffers (apples to apples with gen_step)
            Ke = 8
            eenv = GeneralsEnv(cfg, device=dev, k_slots=Ke, digest=False, actions_out=False)
            eenv.reset()
            eenv.rollout(Ke, 1)
            n_roll = max(2, K // Ke)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(n_roll):
                eenv.rollout(Ke, 1)
            e1.record()
            torch.cuda.synchronize()
            out["rollout_K8_every_step"] = {"env_steps_per_s": N * Ke * n_roll / (e0.elapsed_time(e1) * 1e-3),
                                            "us_per_launch": 1e3 * e0.elapsed_time(e1) / n_roll,
                                            "hbm_frac": N * Ke * (bmin - 4 * H * W * (Ke - 1) / Ke) /
                                                        (e0.elapsed_time(e1) / n_roll * 1e-3) / 1e9 / peak}
            del eenv
            torch.cuda.empty_cache()
        if name == "c3_sweep" and not packed:
            renv = GeneralsEnv(cfg, device=dev, digest=True, actions_out=False)
            renv.reset()
            renv.rollout(32, OBS_DIGEST)
            n_roll = max(2, K // 32)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(n_roll):
                renv.rollout(32, OBS_DIGEST)
            e1.record()
            torch.cuda.synchronize()
            out["rollout_K32_digest"] = {"env_steps_per_s": N * 32 * n_roll / (e0.elapsed_time(e1) * 1e-3),
                                         "us_per_launch": 1e3 * e0.elapsed_time(e1) / n_roll}
            del renv
            torch.cuda.empty_cache()
        print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ NEXT-1: features
def feature_bytes_per_game(H, W, bf16=False, P=2):
    """Algorithmic bytes of one gen_features call per game: per cell read the three state
    planes (4 B) and, per player, write 38 float32 channels (152 B; 76 B as bfloat16, R37), write this turn's two
    history frames (4 B), read the seven previous ones (28 B) and the memory (bits 1 B, last army 2 B, last sighting 4 B)."""
    return H * W * (4 + P * ((76 if bf16 else 152) + 4 + 28 + 7))


def run_features(args):
    """gen_features alone and gen_step + gen_features per turn on BASELINE config 2 (one JSON
    line; not the driver's contract line)."""
    import torch
    import workloads
    from paper_2606_23348_b200 import GeneralsEnv
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, peak_src = measured_peak()
    wl = args.workload or WORKLOAD
    cfg, _ = workloads.config(wl)
    if args.games:
        cfg["n_games"] = args.games
    N, H, W = cfg["n_games"], cfg["height"], cfg["width"]
    K, Wm = args.steps, max(args.warmup, 8)
    bf16 = args.bf16
    env = GeneralsEnv(cfg, device=dev, digest=False, actions_out=False)
    env.reset()
    env.features(bf16=bf16)
    for _ in range(Wm):                       # a full delta history (7 frames) before anything is timed
        env.step()
        env.features()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(K):
        env.step()
        env.features()
    e1.record()
    torch.cuda.synchronize()
    both_ms = e0.elapsed_time(e1) / K
    # the featuriser alone: one event pair per launch (a step in between keeps the contract of one call per turn)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for a, b in ev:
        env.step()
        a.record()
        env.features()
        b.record()
    torch.cuda.synchronize()
    feat_ms = statistics.mean(a.elapsed_time(b) for a, b in ev)
    bfeat = feature_bytes_per_game(H, W, bf16, cfg["n_players"])
    achieved = N * bfeat / (feat_ms * 1e-3) / 1e9
    line = {"workload": f"{wl}: {cfg['n_players']} players {H}x{W}, {N} games, gen_step + gen_features every turn",
            "n_games": N, "steps": K, "dtype": "bf16 (R37)" if bf16 else "f32",
            "feature_tensor_bytes": N * cfg["n_players"] * 38 * env.S * (2 if bf16 else 4),
            "step_plus_features": {"env_steps_per_s": N / (both_ms * 1e-3), "us_per_turn": 1e3 * both_ms},
            "features": {"games_per_s": N / (feat_ms * 1e-3), "us_per_launch": 1e3 * feat_ms,
                         "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                                      "frac": achieved / peak, "traffic": None if bf16 else NCU_FEAT_DRAM_BYTES_PER_LAUNCH.get(N),
                                      "kernel": "gen::k_features" if cfg["n_players"] == 2 else "gen::k_features_mp",
                                      "peak_source": peak_src, "algorithmic_bytes_per_game": bfeat,
                                      "units_per_launch": N}}}
    if not args.no_cpu_baseline:
        from oracle import oracle
        sample, steps = 64, 100
        o = oracle.Oracle(dict(cfg, n_games=sample))
        o.reset()
        o.features()
        t_feat = 0.0
        for _ in range(steps):
            o.step()
            t0 = time.perf_counter()
            o.features()
            t_feat += time.perf_counter() - t0
        line["cpu_baseline"] = {"value": sample * steps / t_feat, "unit": "games/s (orc_features alone)", "cores": 1,
                                "kind": "oracle", "sample": f"first {sample} global game ids x {steps} turns"}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--games", type=int, default=0, help="override games per GPU (default: config 2's 16,384)")
    ap.add_argument("--replicas", type=int, default=0, help="replicas in the round-robin (default: enough for 640 MB)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-large", action="store_true", help="skip the N = 262,144 leg (roofline_large)")
    ap.add_argument("--no-phase-mix", action="store_true", help="headline rotation: every replica starts at turn 0")
    ap.add_argument("--force-step", action="store_true", help="with --only step: k_step also for more than 4 players")
    ap.add_argument("--only", choices=["rollout", "step", "step-large", "rotation", "noalloc"], default="",
                    help="one leg by itself, a few launches (the command of the ncu captures under profiles/)")
    ap.add_argument("--sweep", action="store_true", help="config-3 batch sweep + configs 4 / 5 rows (one JSON line each)")
    ap.add_argument("--rows", default="", help="with --sweep: only the rows whose workload name contains this")
    ap.add_argument("--workload", default="", help="with --features / --only: workload name (default c2_24x24)")
    ap.add_argument("--bf16", action="store_true", help="with --features: the bfloat16 feature tensor (R37)")
    ap.add_argument("--features", action="store_true", help="NEXT-1: gen_features alone and with gen_step (one JSON line)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.only:
        return run_single_leg(args)
    if args.sweep:
        return run_sweep(args)
    if args.features:
        return run_features(args)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
