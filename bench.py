#!/usr/bin/env python
"""bench.py — Stratego env steps/s (legal mask + uniform action + step + bf16 encode) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference]

A "step" is one fused pass of the whole hot path (strat_rollout_step) over one batch of
synthetic games: BASELINE.json configs[2] (classic Stratego, 65,536 games per GPU, 1000-ply
draw cap, auto-reset, Philox-seeded setups, uniform-random legal play).  One JSON line is
printed by rank 0.  `--impl reference` times the CPU oracle instead.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2511_07312_b200 import workloads as W  # noqa: E402

METRIC = "stratego_env_steps_per_sec"
UNIT = "env_steps/s"
ALGO_BYTES_PER_GAME_STEP = 128 + 128 + 452 + 2 + 1 + 1 + 8800  # state R+W, mask, action, reward, done, obs = 9512
CFG = W.CONFIGS[2]


def ncu_constant(kernel, key):
    """Per-launch counters taken from an `ncu --set full` capture (profiles/ncu_constants.json
    names the capture, its command and the commit the kernel was at).  None if not recorded."""
    try:
        rec = json.load(open(os.path.join(ROOT, "profiles", "ncu_constants.json")))[kernel]
        return rec.get(key), "%s @ %s" % (rec.get("source"), rec.get("commit"))
    except Exception:
        return None, None


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.005)

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def oracle_rate(num_games, steps, warmup):
    """The oracle as it stands on one host core: config-2 shape on `num_games` games."""
    from oracle import orc
    e = orc.Env(num_games, variant=CFG["variant"], seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1)

    def one():
        m = e.legal_mask()
        a = e.sample_uniform(m)
        e.step(a)
        e.encode_obs()

    for _ in range(warmup):
        one()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    dt = time.perf_counter() - t0
    return num_games * steps / dt, dt


def _oracle_shard(q, num_games, steps, warmup, base):
    from oracle import orc
    e = orc.Env(num_games, variant=CFG["variant"], seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1,
                game_base=base)

    def one():
        e.step(e.sample_uniform(e.legal_mask()))
        e.encode_obs()

    for _ in range(warmup):
        one()
    q.put("ready")
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    q.put(time.perf_counter() - t0)


def oracle_rate_all_cores(num_games, steps, warmup):
    """The same oracle as independent game shards, one process per host core (no tuning): total
    game-steps / the slowest shard's time."""
    import multiprocessing as mp
    cores = host_cores()
    ctx = mp.get_context("spawn")
    qs, ps = [], []
    for k in range(cores):
        q = ctx.Queue()
        p = ctx.Process(target=_oracle_shard, args=(q, num_games, steps, warmup, k * num_games), daemon=True)
        p.start()
        qs.append(q); ps.append(p)
    for q in qs:
        q.get()
    t0 = time.perf_counter()
    times = [q.get() for q in qs]
    wall = time.perf_counter() - t0
    for p in ps:
        p.join(timeout=10)
    return cores * num_games * steps / max(max(times), 1e-9), cores, wall


def launch_ranks(args):
    """`python bench.py --gpus N` with N > 1 and no launcher around it (the paper
    runs 16 data-parallel GPUs): start N ranks of this same command line under
    torch.distributed.run on 127.0.0.1, one per GPU, and hand back its exit code.  Every rank then runs
    main() again with WORLD_SIZE set and takes the sharded path."""
    import socket
    import subprocess
    if args.impl == "b200":
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit("bench.py: --gpus %d but this node has %d CUDA device(s)" % (args.gpus, have))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:  # every rank reports in (gloo, CPU), then rank 0 alone works and prints
        import torch
        import torch.distributed as dist
        dist.init_process_group("gloo")
        seen = torch.ones(1, dtype=torch.int64)
        dist.all_reduce(seen)
        dist.destroy_process_group()
        world = int(seen.item())
    if rank != 0:
        return
    # each step = one pass of the oracle over a bounded sample of the 65,536-game workload,
    # sized so the whole run takes ~20 s at ~16k game-steps/s/core
    total = args.steps + args.warmup
    games = max(32, min(CFG["num_games"], 320000 // max(total, 1)))
    rate, dt = oracle_rate(games, args.steps, args.warmup)
    sample = "%d of %d games per step (same seed, global game indices 0..%d), %d steps" % (
        games, CFG["num_games"], games - 1, args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1000.0 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": CFG["name"], "games_per_step": games, "parallelism": "1 host core", "ranks_started": world},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_e2e(args, env, B, torch, dist, world, barrier, stream, mask, act, rew, done):
    """End to end through the host-buffer C-ABI call strat_step_host (max over ranks)."""
    n = env.n
    e2e_steps = max(3, min(args.steps, 12))
    env.reset(CFG["seed"])
    rec = torch.empty((args.warmup + e2e_steps, n), dtype=torch.int16).pin_memory()
    for k in range(args.warmup + e2e_steps):  # record a legal action sequence (deterministic replay)
        m = env.legal_mask(mask)
        a = env.sample_uniform(m, act)
        rec[k].copy_(a, non_blocking=False)
        env.step(a, rew, done)
    env.reset(CFG["seed"])
    scratch = env.host_scratch()
    h_rew = torch.empty(n, dtype=torch.int8).pin_memory()
    h_done = torch.empty(n, dtype=torch.uint8).pin_memory()
    h_mask = torch.empty((n, 113), dtype=torch.int32).pin_memory()
    h_obs = torch.empty((n, 4400), dtype=torch.bfloat16).pin_memory()
    for k in range(args.warmup):
        env.step_host(scratch, rec[k], h_rew, h_done, h_mask, h_obs)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(e2e_steps):
        env.step_host(scratch, rec[args.warmup + k], h_rew, h_done, h_mask, h_obs)
    e1.record(stream)
    barrier()
    assert env.check() == 0
    t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return world * n * e2e_steps / (float(t.item()) / 1e3), e2e_steps



def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2511_07312_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA device required (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    n = CFG["num_games"]
    kw = W.shard_for_rank(CFG, rank, world)  # weak scaling: n independent games per rank, no data-path collective
    kw["device"] = local
    kw["chase_rule"] = 1 if args.chase_rule else 0
    env = B.Env(n, **kw)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # Steady state (BASELINE.json configs[2]: "measure the steady-state rate"): all games start at ply 0 in
    # lockstep and the mean game lasts ~560 plies, so a short run would time young, synchronised games only.
    # 1,500 on-chip plies with auto-reset (strat_rollout_uniform = that many mask + sample + step passes,
    # ~7 ms) desynchronise them before the warm-up, whatever --steps / --warmup are.
    PRE_AGE_PLIES = 1500
    env.rollout_uniform(PRE_AGE_PLIES)
    for _ in range(args.warmup):
        env.rollout_step(mask, act, rew, done, obs)
    b0 = env.get_boards()
    window_start_ply_mean = float((b0[:, 116].to(torch.float64) + 256.0 * b0[:, 117].to(torch.float64)).mean().item())
    del b0
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    # Consecutive fused steps overlap on the device (programmatic dependent launch) and an event
    # record between two launches serialises them: events at the two ends of the timed region,
    # plus interior marks at least 50 launches apart (none below 100 steps).
    chunk = max(50, args.steps // 20)
    marks = (list(range(0, args.steps - chunk + 1, chunk)) if args.steps >= 100 else [0]) + [args.steps]
    ev = [torch.cuda.Event(enable_timing=True) for _ in marks]
    ev[0].record(stream)
    nxt = 1
    for k in range(args.steps):
        env.rollout_step(mask, act, rew, done, obs)
        if k + 1 == marks[nxt]:
            ev[nxt].record(stream)
            nxt += 1
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = sorted(ev[i].elapsed_time(ev[i + 1]) / (marks[i + 1] - marks[i]) for i in range(len(marks) - 1))
    median_ms = per_step[len(per_step) // 2] if len(per_step) >= 3 else None
    assert env.check() == 0
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    value = world * n * args.steps / (total_ms_max / 1e3)
    per_rank_ms = [total_ms / args.steps]
    if world > 1:
        mine = torch.tensor([total_ms / args.steps], dtype=torch.float64, device="cuda")
        every = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(every, mine)
        per_rank_ms = [float(x.item()) for x in every]

    # outside the timed region (the steps that follow it): sanity statistics of the workload
    # (SURVEY.md section 5 "Metrics"): games ended per step, why, how long they were, legal moves
    stat_steps = 50
    popc = torch.tensor([bin(i).count("1") for i in range(256)], dtype=torch.int64, device="cuda")
    ended, legal_sum, len_sum = 0, 0, 0
    reasons = torch.zeros(8, dtype=torch.int64, device="cuda")
    for _ in range(stat_steps):
        b = env.get_boards()
        ply = b[:, 116].to(torch.int64) | (b[:, 117].to(torch.int64) << 8)
        env.rollout_step(mask, act, rew, done, obs)
        fin = (done & 1).bool()
        ended += int(fin.sum().item())
        len_sum += int((ply[fin] + 1).sum().item())
        reasons += torch.bincount(((done[fin] >> 2) & 7).to(torch.int64), minlength=8)
        legal_sum += int(popc[mask.view(torch.uint8).to(torch.int64)].sum().item())
    reset_fraction = ended / float(stat_steps * n)
    reason_names = ["", "flag_captured", "no_move_win", "no_move_draw", "ply_cap", "battleless"]
    stats = {"window": "%d steps after the timed region" % stat_steps, "games_ended": ended,
             "pre_aged_plies": PRE_AGE_PLIES, "window_start_ply_mean": window_start_ply_mean,
             "termination_reasons": {reason_names[k]: int(reasons[k].item()) for k in range(1, 6)},
             "mean_game_length_plies": (len_sum / ended) if ended else None,
             "mean_legal_moves": legal_sum / float(stat_steps * n)}

    # Two side measurements, outside the timed region.  (1) The same loop writing into 4 rotating sets of
    # output buffers: consecutive steps then never hit each other's lines in the L2 (with one set, ~4 % of a
    # step's output is overwritten there before it reaches DRAM, profiles/r2_rollout_step_range.md).
    # (2) The plain-write figure of this GPU for the store instruction the kernel uses, in batch-sized pieces
    # handed out by ticket (as the kernel does) and in equal shares (strat_probe_write).
    rot_sets, rot_steps = 4, max(50, min(args.steps, 400))
    sets = [(env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()) for _ in range(rot_sets - 1)]
    sets.append((mask, act, rew, done, obs))
    for k in range(20):
        env.rollout_step(*sets[k % rot_sets])
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0.record(stream)
    for k in range(rot_steps):
        env.rollout_step(*sets[k % rot_sets])
    r1.record(stream)
    torch.cuda.synchronize()
    rot_ms = r0.elapsed_time(r1) / rot_steps
    del sets
    probe = torch.empty(n * 8800, dtype=torch.uint8, device="cuda")  # one step's observations
    ceil = {}
    for name, dyn in (("by_ticket", True), ("equal_shares", False)):
        for _ in range(5):
            env.probe_write(probe, 281600, dyn)
        r0.record(stream)
        for _ in range(40):
            env.probe_write(probe, 281600, dyn)
        r1.record(stream)
        torch.cuda.synchronize()
        ceil[name] = probe.numel() * 40 / (r0.elapsed_time(r1) / 1e3) / 1e9
    del probe
    assert env.check() == 0

    e2e_value, e2e_steps = None, 0
    if not args.skip_e2e:
        e2e_value, e2e_steps = run_e2e(args, env, B, torch, dist, world, barrier, stream, mask, act, rew, done)
    if rank == 0:
        peak, peak_src = measured_peak_gbs()
        kernel_ms = total_ms / args.steps  # the step IS one launch of k_rollout_step
        achieved = ALGO_BYTES_PER_GAME_STEP * n / (kernel_ms / 1e3) / 1e9
        cpu_games, cpu_steps = 2048, 150
        cpu_rate, cpu_dt = oracle_rate(cpu_games, cpu_steps, 10) if (world == 1 and not args.skip_cpu) else (None, None)
        all_rate = all_cores = all_wall = None
        if cpu_rate is not None:
            all_rate, all_cores, all_wall = oracle_rate_all_cores(1024, 150, 5)
        frac = achieved / peak
        traffic, traffic_src = ncu_constant("k_rollout_step", "dram_bytes_per_launch") if n == 65536 else (None, None)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms_max / args.steps, "median_ms_per_step": median_ms, "higher_is_better": True,
            "ms_per_step_per_rank": per_rank_ms,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": CFG["name"], "games_per_gpu": n, "variant": "classic", "max_plies": CFG["max_plies"],
                       "auto_reset": 1, "chase_rule": 1 if args.chase_rule else 0,
                       "games_reset_per_step_fraction": reset_fraction, "stats": stats,
                       "event_marks": len(marks),
                       "rotating_outputs": {"sets": rot_sets, "steps": rot_steps, "ms_per_step": rot_ms,
                                            "achieved_gbs": ALGO_BYTES_PER_GAME_STEP * n / (rot_ms / 1e3) / 1e9},
                       "policy": "uniform-random legal (Philox4x32-10)",
                       "parallelism": "games sharded over %d GPU(s), no collective" % world,
                       "l2": "outputs 623 MB/step per GPU > 126 MB L2 (no flush needed)"},
            "roofline": {"bound": "hbm", "kernel": "k_rollout_step", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": frac, "traffic": traffic,
                         "traffic_source": traffic_src,
                         "peak_source": peak_src,
                         "note": ("peak is a measured copy (half reads, half writes); this kernel is a write stream "
                                  "whose batches are handed out by ticket and exceeds it, hence frac > 1: see "
                                  "write_ceiling") if frac > 1.0 else
                                 "peak is a measured copy (half reads, half writes)",
                         "write_ceiling": {"unit": "GB/s", "by_ticket": ceil["by_ticket"], "equal_shares": ceil["equal_shares"],
                                           "how": "strat_probe_write: 16-byte st.global.cs over one step's observations "
                                                  "(%d MB) in 281,600-byte pieces, 40 launches" % (n * 8800 // 1000000)},
                         "frac_of_write_ceiling": achieved / ceil["by_ticket"],
                         "algorithmic_bytes_per_game_step": ALGO_BYTES_PER_GAME_STEP,
                         "frac_of_nominal_8000": achieved / 8000.0},
            "e2e": None if e2e_value is None else {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * n * world,
                    "d2h_bytes_per_step": (8800 + 452 + 1 + 1) * n * world, "steps": e2e_steps,
                    "call": "strat_step_host (pinned host actions in; reward, done, next mask, next obs out)"},
            "gpu_launches": args.steps,
            "clocks": sampler.result(),
        }
        if cpu_rate is not None:
            line["cpu_baseline"] = {"value": cpu_rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": "%d games x %d steps of the same workload (%.1f s)" % (cpu_games, cpu_steps, cpu_dt),
                                    "host_cores": host_cores(),
                                    "all_cores": {"value": all_rate, "unit": UNIT, "cores": all_cores,
                                                  "sample": "independent shards of 1024 games x 150 steps, one oracle process "
                                                            "per host core (%.1f s)" % all_wall}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_profile_range(args):
    """The overlapped regime under ncu's range replay: K consecutive launches of the fused step in
    one profiled range (they run concurrently as they do in production; per-kernel replay would
    serialise them).  A number printed by a run under a profiler is not a bench value."""
    import torch
    from paper_2511_07312_b200 import binding as B
    n = CFG["num_games"]
    env = B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1,
                chase_rule=1 if args.chase_rule else 0)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    for _ in range(max(args.warmup, 20)):
        env.rollout_step(mask, act, rew, done, obs)
    torch.cuda.synchronize()
    rt = torch.cuda.cudart()
    rt.cudaProfilerStart()
    for _ in range(args.profile_range):
        env.rollout_step(mask, act, rew, done, obs)
    torch.cuda.synchronize()
    rt.cudaProfilerStop()
    assert env.check() == 0
    print(json.dumps({"profile_range": args.profile_range, "games_per_launch": n,
                      "algorithmic_bytes_per_launch": ALGO_BYTES_PER_GAME_STEP * n}))


def _peak_line(achieved):
    peak, src = measured_peak_gbs()
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": None, "peak_source": src, "frac_of_nominal_8000": achieved / 8000.0}


def run_cfg3(args):
    """BASELINE.json configs[3]: 262,144 games; every step also appends the transition to a
    64 x 131,072-record device ring (zero-copy: the fused step writes mask_t and obs_{t+1} in
    place) and gathers a uniform 4,096-transition minibatch."""
    import torch
    from paper_2511_07312_b200 import binding as B
    c = W.CONFIGS[3]
    n = c["num_games"]
    env = B.Env(n, variant=0, seed=c["seed"], max_plies=c["max_plies"], auto_reset=1)
    ring = B.Replay(c["ring_per_slot"], c["ring_slots"], block=n)  # spare rows: nothing written ahead is live
    act, rew, done = env.new_actions(), env.new_reward(), env.new_done()
    bs = c["sample_batch"]
    s_obs = torch.empty((bs, 44, 10, 10), dtype=torch.bfloat16, device="cuda")
    s_mask = torch.empty((bs, 113), dtype=torch.int32, device="cuda")
    s_act = torch.empty(bs, dtype=torch.int16, device="cuda")
    s_rew = torch.empty(bs, dtype=torch.int8, device="cuda")
    s_done = torch.empty(bs, dtype=torch.uint8, device="cuda")
    o_ptr, _ = ring.reserve(n, 0)
    B._chk(B.lib().strat_encode_obs(env.h, o_ptr, B._stream()), "encode")

    def step(t):
        _, m_ptr = ring.reserve(n, 0)
        o_next, _ = ring.reserve(n, 1)
        a_ptr, r_ptr, d_ptr = ring.reserve_rows(n)
        env.rollout_step_ptrs(m_ptr, a_ptr, r_ptr, d_ptr, o_next)  # all five arrays written in place
        ring.commit_in_place(n)                                     # host bookkeeping only
        # chained gather: the next fused step still overlaps this one on the device
        ring.sample_chained(env, c["seed"], t, bs, s_obs, s_mask, s_act, s_rew, s_done)

    for t in range(args.warmup):
        step(t)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for t in range(args.steps):
        step(args.warmup + t)
    e1.record()
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    assert env.check() == 0
    ms = e0.elapsed_time(e1)
    per_game = ALGO_BYTES_PER_GAME_STEP + 2 * bs * W.TRANSITION_BYTES / n  # + gather R/W
    line = {
        "metric": METRIC, "value": n * args.steps / (ms / 1e3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": c["name"], "games_per_gpu": n, "ring": "%d x %d records, %.1f GB" % (
            c["ring_slots"], c["ring_per_slot"], ring.mem.numel() / 1e9), "sample_batch": bs,
            "push": "zero-copy (fused step writes mask_t, action_t, reward_t, done_t, obs_t+1 into the ring rows)"},
        "roofline": dict(_peak_line(per_game * n / (ms / args.steps / 1e3) / 1e9), kernel="k_rollout_step + k_replay_sample",
                         algorithmic_bytes_per_game_step=per_game),
        "gpu_launches": 2 * args.steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def cfg4_roofline(ms_rollout):
    inst, src = ncu_constant("k_rollout_uniform", "warp_inst_per_launch")
    traffic, _ = ncu_constant("k_rollout_uniform", "dram_bytes_per_launch")
    peak = 148 * 4 * 1.965
    ach = None if inst is None else inst / (ms_rollout / 1e3) / 1e9
    return {"bound": "alu", "kernel": "k_rollout_uniform", "achieved": ach, "peak": peak, "unit": "G warp-inst/s",
            "frac": None if ach is None else ach / peak, "traffic": traffic, "source": src}


def run_cfg4(args):
    """BASELINE.json configs[4]: 16 roots (ply 200) x 16,384 determinisations, 64-ply uniform
    rollouts with the boards on chip, per-root reduction.  A 'step' = the whole batch."""
    import numpy as np
    import torch
    from paper_2511_07312_b200 import binding as B
    c = W.CONFIGS[4]
    R, S, plies = c["num_roots"], c["samples_per_root"], c["rollout_plies"]
    src = B.Env(R, variant=0, seed=c["seed"], max_plies=1000, auto_reset=1)

    def play():
        src.step(src.sample_uniform(src.legal_mask()))

    rb = W.capture_at_ply(lambda: src.get_boards().cpu().numpy(), play, R, c["root_plies"])
    roots = B.Env(R, variant=0, seed=c["seed"])
    roots.reset_from(torch.from_numpy(rb).cuda())
    side = torch.from_numpy(((rb[:, 116].astype(np.int64) | (rb[:, 117].astype(np.int64) << 8)) & 1).astype(np.uint8)).cuda()
    out = B.Env(R * S, variant=0, seed=c["seed"], max_plies=0, auto_reset=0)
    red = torch.empty((R, 3), dtype=torch.int32, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    t_det = t_roll = t_red = 0.0
    steps = max(1, min(args.steps, 20))
    sampler = ClockSampler(0)
    sampler.start()
    for k in range(min(args.warmup, 3) + steps):
        ev[0].record()
        B.determinise(roots, S, 1000 + k, out)
        ev[1].record()
        out.rollout_uniform(plies)
        ev[2].record()
        B.reduce_returns(out, side, S, red)
        ev[3].record()
        torch.cuda.synchronize()
        if k >= min(args.warmup, 3):
            t_det += ev[0].elapsed_time(ev[1]); t_roll += ev[1].elapsed_time(ev[2]); t_red += ev[2].elapsed_time(ev[3])
    sampler.stop_flag = True
    sampler.join()
    assert out.check() == 0 and roots.check() == 0
    total = t_det + t_roll + t_red
    line = {
        "metric": METRIC, "value": R * S * plies * steps / (total / 1e3), "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": min(args.warmup, 3), "ms_per_step": total / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": c["name"], "roots": R, "samples_per_root": S, "rollout_plies": plies,
                   "ms_determinise": t_det / steps, "ms_rollout": t_roll / steps, "ms_reduce": t_red / steps,
                   "rollout_env_steps_per_sec": R * S * plies * steps / (t_roll / 1e3),
                   "note": "ALU/latency-bound: boards stay in registers for all 64 plies (256 B of HBM per game)",
                   "returns_sum_wins_losses_root0": red[0].tolist()},
        # instruction-issue bound: peak = SMs x 4 schedulers x 1 warp instruction per clock x max SM clock
        # (DESIGN.md section 6); achieved = ncu smsp__inst_executed.sum of one rollout launch / its CUDA-event time
        "roofline": cfg4_roofline(t_roll / steps),
        "gpu_launches": 3 * steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_search(args):
    """One network-free search step per root (Table S12: 1,000 rollouts of depth
    40 over sampled configurations x legal actions, forced first move, eq. 8) for 256 roots at
    once; uniform policy / game result stand in for the move network's policy / value."""
    import numpy as np
    import torch
    from paper_2511_07312_b200 import binding as B
    R, rollouts, depth = 256, 1000, 40
    src = B.Env(R, variant=0, seed=0, max_plies=1000, auto_reset=1)
    rb = W.capture_at_ply(lambda: src.get_boards().cpu().numpy(), lambda: src.step(src.sample_uniform(src.legal_mask())), R, 200)
    roots = B.Env(R, variant=0, seed=0)
    roots.reset_from(torch.from_numpy(rb).cuda())
    games = B.Env(R * rollouts, variant=0, seed=0, max_plies=0, auto_reset=0)
    outs = tuple(torch.empty((R, 3600), dtype=torch.float32, device="cuda") for _ in range(3))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    steps = max(1, min(args.steps, 20))
    sampler = ClockSampler(0)
    sampler.start()
    t = [0.0, 0.0, 0.0]
    for k in range(min(args.warmup, 3) + steps):
        ev[0].record()
        B.search_expand(roots, rollouts, 500 + k, games)
        ev[1].record()
        games.rollout_uniform(depth - 1)
        ev[2].record()
        B.search_policy(roots, games, rollouts, 0.002, 0.02, None, outs)
        ev[3].record()
        torch.cuda.synchronize()
        if k >= min(args.warmup, 3):
            for i in range(3):
                t[i] += ev[i].elapsed_time(ev[i + 1])
    sampler.stop_flag = True
    sampler.join()
    assert games.check() == 0 and roots.check() == 0
    total = sum(t)
    legal = (outs[2] > 0).sum(dim=1).float().mean().item()
    line = {
        "metric": METRIC, "value": R * rollouts * depth * steps / (total / 1e3), "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": min(args.warmup, 3), "ms_per_step": total / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8 (game), f32 (eq. 8)", "data": "synthetic",
        "config": {"workload": "search_step_256_roots", "roots": R, "rollouts_per_root": rollouts, "depth": depth,
                   "ms_expand": t[0] / steps, "ms_rollout": t[1] / steps, "ms_policy": t[2] / steps,
                   "searched_moves_per_sec": R * steps / (total / 1e3), "mean_legal_actions": legal,
                   "note": "env-step count includes unused slots' share (rollouts*depth per root); paper: 1.26 s per "
                           "searched move on one H100 WITH its networks (PAPER.md:200) - context only"},
        "gpu_launches": 3 * steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_infostate(args):
    """The paper's own information state on the headline shape (PAPER.md:462, S2 482-610): 65,536
    classic games; every step = one fused step that also keeps the S2 trackers up to date, then
    ComputeInfostateTensor in the 487-channel bf16 form (97,400 bytes per game) for every game."""
    import torch
    from paper_2511_07312_b200 import binding as B
    n = CFG["num_games"]
    env = B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], max_battleless=200, auto_reset=1, infostate=1)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    info = env.new_infostate()
    steps = max(1, min(args.steps, 200))
    for _ in range(max(args.warmup, 3)):
        env.rollout_step(mask, act, rew, done, obs)
        env.encode_infostate(info)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    for k in range(steps):
        ev[k][0].record()
        env.rollout_step(mask, act, rew, done, obs)
        ev[k][1].record()
        env.encode_infostate(info)
        ev[k][2].record()
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    assert env.check() == 0
    ms_step = sum(e[0].elapsed_time(e[1]) for e in ev) / steps
    ms_enc = sum(e[1].elapsed_time(e[2]) for e in ev) / steps
    total = ev[0][0].elapsed_time(ev[-1][2]) / steps
    per_game = 487 * 100 * 2 + 2048 + 128  # the tensor out, the tracker block and the line in
    line = {
        "metric": "stratego_infostates_per_sec", "value": n / (total / 1e3), "unit": "information states/s", "n_gpus": 1,
        "steps": steps, "warmup": max(args.warmup, 3), "ms_per_step": total, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8 (game), bf16 (tensor; real-valued channels rounded once from f64)", "data": "synthetic",
        "config": {"workload": CFG["name"] + " + 487-channel information state", "games_per_gpu": n,
                   "ms_tracked_fused_step": ms_step, "ms_encode_infostate": ms_enc,
                   "tensor_bytes_per_game": 487 * 100 * 2, "tracker_bytes_per_game": 2048,
                   "l2": "output 6.38 GB per step > 126 MB L2 (no flush needed)"},
        "roofline": dict(_peak_line(per_game * n / (ms_enc / 1e3) / 1e9), kernel="k_encode_infostate",
                         algorithmic_bytes_per_game=per_game, traffic=ncu_constant("k_encode_infostate", "dram_bytes_per_launch")[0],
                         traffic_source=ncu_constant("k_encode_infostate", "dram_bytes_per_launch")[1]),
        "gpu_launches": 2 * steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_observe(args):
    """The data-collection loop with an external policy: a policy kernel
    picks the actions from the mask (here the uniform sampler stands in for the move network), then
    strat_step_observe applies them and writes mask + observation of the new state in one pass.  The
    fused step cannot overlap its neighbours here: it is timed as an isolated launch."""
    import torch
    from paper_2511_07312_b200 import binding as B
    n = CFG["num_games"]
    env = B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    env.legal_mask(mask)
    steps = max(1, min(args.steps, 500))
    for _ in range(max(args.warmup, 3)):
        env.sample_uniform(mask, act)
        env.step_observe(act, rew, done, mask, obs)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    for k in range(steps):
        ev[k][0].record()
        env.sample_uniform(mask, act)
        ev[k][1].record()
        env.step_observe(act, rew, done, mask, obs)
        ev[k][2].record()
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    assert env.check() == 0
    ms_pol = sorted(e[0].elapsed_time(e[1]) for e in ev)[steps // 2]
    ms_obs = sorted(e[1].elapsed_time(e[2]) for e in ev)[steps // 2]
    total = ev[0][0].elapsed_time(ev[-1][2]) / steps
    line = {
        "metric": METRIC, "value": n / (total / 1e3), "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": CFG["name"] + " with an external policy kernel", "games_per_gpu": n,
                   "ms_policy_stand_in": ms_pol, "ms_step_observe_median": ms_obs,
                   "note": "events between the two kernels: strat_step_observe is timed as an isolated launch"},
        "roofline": dict(_peak_line(ALGO_BYTES_PER_GAME_STEP * n / (ms_obs / 1e3) / 1e9), kernel="k_rollout_step<external>",
                         algorithmic_bytes_per_game_step=ALGO_BYTES_PER_GAME_STEP,
                         traffic=ncu_constant("k_rollout_step_observe", "dram_bytes_per_launch")[0],
                         traffic_source=ncu_constant("k_rollout_step_observe", "dram_bytes_per_launch")[1]),
        "gpu_launches": 2 * steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_observe2(args):
    """A usage-level answer to the lone-launch gap of `observe` (an isolated strat_step_observe ends unevenly and
    the write stream drains between launches): the same 65,536 games as TWO environments of 32,768 on two streams,
    each running policy stand-in -> strat_step_observe.  One environment's step then runs while the other's policy
    kernel (and launch head / tail) does, so the HBM write stream need not drain.  Reports the pair's rate."""
    import torch
    from paper_2511_07312_b200 import binding as B
    n = CFG["num_games"] // 2
    envs = [B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1, game_base=k * n) for k in (0, 1)]
    bufs = [(e.new_mask(), e.new_actions(), e.new_reward(), e.new_done(), e.new_obs()) for e in envs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for e, (mask, act, rew, done, obs) in zip(envs, bufs):
        e.rollout_uniform(1500)   # desynchronised games, as in the headline run
        e.legal_mask(mask)
    torch.cuda.synchronize()
    steps, warm = max(1, min(args.steps, 1000)), max(args.warmup, 3)

    def loop_interleaved(k):   # issue order alternates between the streams, as one host thread driving both would
        for _ in range(k):
            for e, st, (mask, act, rew, done, obs) in zip(envs, streams, bufs):
                with torch.cuda.stream(st):
                    e.sample_uniform(mask, act)
                    e.step_observe(act, rew, done, mask, obs)

    loop_interleaved(warm)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    cur = torch.cuda.current_stream()
    e0.record(cur)
    for st in streams:
        st.wait_event(e0)
    loop_interleaved(steps)
    for st in streams:
        cur.wait_stream(st)
    e1.record(cur)
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    for e in envs:
        assert e.check() == 0
    ms = e0.elapsed_time(e1) / steps   # one step of BOTH environments = 65,536 game-steps
    line = {
        "metric": METRIC, "value": 2 * n / (ms / 1e3), "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": warm,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": CFG["name"] + " as two 32,768-game environments on two streams, external policy kernel",
                   "games_per_gpu": 2 * n, "environments": 2,
                   "note": "per step and environment: policy stand-in (strat_sample_uniform) then strat_step_observe; "
                           "the two streams are only ordered at the ends of the timed region",
                   "l2": "outputs 623 MB per step of the pair > 126 MB L2 (no flush needed)"},
        "roofline": dict(_peak_line(ALGO_BYTES_PER_GAME_STEP * 2 * n / (ms / 1e3) / 1e9), kernel="k_rollout_step<external> x 2 streams",
                         algorithmic_bytes_per_game_step=ALGO_BYTES_PER_GAME_STEP),
        "gpu_launches": 4 * steps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_small(args, idx):
    """BASELINE.json configs[0] (256 classic games, 256 plies) and configs[1] (4,096 Barrage games to
    termination, 2,000-ply draw cap): report-only lines.  Both are far too small to
    load the GPU (2.4 MB / 39 MB of output per step against 623 MB for the headline): the rate is set by
    the launch, not by HBM.  A step is one fused pass (strat_rollout_step) over all games, finished ones
    included (no auto-reset in these configs: they stay frozen and emit empty masks)."""
    import torch
    from paper_2511_07312_b200 import binding as B
    cfg = W.CONFIGS[idx]
    n, steps = cfg["num_games"], cfg["steps"]
    kw = dict(variant=cfg["variant"], seed=cfg["seed"], max_plies=cfg["max_plies"], auto_reset=cfg["auto_reset"])
    env = B.Env(n, **kw)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    for _ in range(max(args.warmup, 3)):
        env.rollout_step(mask, act, rew, done, obs)
    reps = max(1, min(args.steps, 20))
    sampler = ClockSampler(0)
    sampler.start()
    times, live_steps = [], 0
    reasons = torch.zeros(8, dtype=torch.int64, device="cuda")
    for r in range(reps):  # every repetition plays the config from its seeded start
        env.reset(cfg["seed"])
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            env.rollout_step(mask, act, rew, done, obs)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    sampler.stop_flag = True
    sampler.join()
    # outside the timed region: one more play-through for the termination histogram and the live game-steps
    env.reset(cfg["seed"])
    for _ in range(steps):
        env.rollout_step(mask, act, rew, done, obs)
        live_steps += int((act >= 0).sum().item())
    flags = env.get_boards()[:, 120]   # final state of every game: bit 0 done, bits 2-4 reason
    fin = (flags & 1).bool()
    reasons += torch.bincount(((flags[fin] >> 2) & 7).to(torch.int64), minlength=8)
    assert env.check() == 0
    ms = sorted(times)[len(times) // 2] / steps
    names = ["", "flag_captured", "no_move_win", "no_move_draw", "ply_cap", "battleless"]
    per_step_bytes = ALGO_BYTES_PER_GAME_STEP * n
    line = {
        "metric": METRIC, "value": n / (ms / 1e3), "unit": UNIT, "n_gpus": 1, "steps": steps * reps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": cfg["name"], "games_per_gpu": n, "plies": steps, "repetitions": reps,
                   "bound": "launch (a step writes %.1f MB; the headline step writes 623 MB in 83 us)" % (per_step_bytes / 1e6),
                   "live_game_steps": live_steps, "live_game_steps_per_sec": live_steps / (ms * steps / 1e3),
                   "games_finished": int(reasons.sum().item()),
                   "termination_reasons": {names[k]: int(reasons[k].item()) for k in range(1, 6)},
                   "l2": "outputs fit the 126 MB L2 at this size: a launch-bound line, not an HBM figure"},
        "roofline": dict(_peak_line(per_step_bytes / (ms / 1e3) / 1e9), kernel="k_rollout_step",
                         algorithmic_bytes_per_game_step=ALGO_BYTES_PER_GAME_STEP),
        "gpu_launches": steps * reps, "clocks": sampler.result(),
    }
    print(json.dumps(line))


def run_hist(args):
    """The paper's own buffer design on the headline workload: the fused step
    records the 128-byte state of every game and step into a 256-step board-history ring
    (2.2 GB instead of 155 GB of stored transitions), and masks / information states of past
    steps are re-materialised on demand."""
    import torch
    from paper_2511_07312_b200 import binding as B
    n, length = CFG["num_games"], 256
    env = B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1)
    hist = B.History(n, length)
    hist_bytes = hist.mem.numel()
    hist.attach(env)
    mask, act, rew, done, obs = env.new_mask(), env.new_actions(), env.new_reward(), env.new_done(), env.new_obs()
    for _ in range(args.warmup):
        env.rollout_step(mask, act, rew, done, obs)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    e[0].record()
    for _ in range(args.steps):
        env.rollout_step(mask, act, rew, done, obs)
    e[1].record()
    cur = hist.current_step()
    q = max(10, min(args.steps, 200))
    for k in range(q):  # re-materialise mask + information state of a past step
        t = cur - 1 - (k * 37) % min(length, cur)
        hist.legal_mask(t, mask)
        hist.encode_obs(t, obs)
    e[2].record()
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    assert env.check() == 0
    ms_step, ms_q = e[0].elapsed_time(e[1]) / args.steps, e[1].elapsed_time(e[2]) / q
    per_game = ALGO_BYTES_PER_GAME_STEP + 128 + 4  # + recorded state line + action/reward/done
    # Side measurement, outside the timed region: the paper's own 487-channel information state of PAST steps
    # (ComputeInfostateTensor(t)) from a tracked ring, which also keeps the 2 KB of S2
    # trackers per game and step (a copy kernel in front of every recorded step).
    del hist, env
    tlen, tsteps, tq = 32, 48, 20
    tenv = B.Env(n, variant=0, seed=CFG["seed"], max_plies=CFG["max_plies"], auto_reset=1, infostate=1)
    thist = B.History(n, tlen, tracked=True)
    thist.attach(tenv)
    for _ in range(8):
        tenv.rollout_step(mask, act, rew, done, obs)
    info = tenv.new_infostate()
    thist.encode_infostate(thist.current_step() - 1, info)
    f = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    f[0].record()
    for _ in range(tsteps):
        tenv.rollout_step(mask, act, rew, done, obs)
    f[1].record()
    tcur = thist.current_step()
    for k in range(tq):
        thist.encode_infostate(tcur - 1 - (k * 7) % tlen, info)
    f[2].record()
    torch.cuda.synchronize()
    assert tenv.check() == 0
    ms_tstep, ms_q487 = f[0].elapsed_time(f[1]) / tsteps, f[1].elapsed_time(f[2]) / tq
    q487_gbs = 97400.0 * n / (ms_q487 / 1e3) / 1e9
    hist487 = dict(_peak_line(q487_gbs), call="strat_history_encode_infostate of a past step", ms_per_query=ms_q487,
                   algorithmic_bytes_per_game=97400, ring_steps=tlen, ring_bytes=thist.mem.numel(),
                   tracker_bytes_per_game_step=2048, ms_per_recorded_tracked_step=ms_tstep)
    line = {
        "metric": METRIC, "value": n / (ms_step / 1e3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": CFG["name"] + " + board-history ring", "games_per_gpu": n, "history_steps": length,
                   "history_bytes": hist_bytes, "historical_infostate487": hist487,
                   "historical_query": "strat_history_legal_mask + strat_history_encode_obs of a past step",
                   "ms_per_historical_query": ms_q, "historical_game_queries_per_sec": n / (ms_q / 1e3)},
        "roofline": dict(_peak_line(per_game * n / (ms_step / 1e3) / 1e9), kernel="k_rollout_step (recording)",
                         algorithmic_bytes_per_game_step=per_game),
        "gpu_launches": args.steps + 2 * q, "clocks": sampler.result(),  # timed region only
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4", "hist", "search", "infostate487", "observe", "observe2"],
                    help="cfg2 = the headline (default); cfg0 / cfg1 = BASELINE.json configs[0] / [1] (report only, launch-bound); "
                         "cfg3 / cfg4 = BASELINE.json configs[3] / [4]; "
                         "hist = cfg2 recording into the board-history ring + historical queries; "
                         "search = network-free search steps (S3.7) for 256 roots; infostate487 = cfg2 with the S2 trackers kept and the "
                         "paper's 487-channel information state encoded every step; observe = cfg2 driven by an external policy "
                         "kernel through strat_step_observe; observe2 = the same games as two environments on two streams; all 1 GPU")
    ap.add_argument("--chase-rule", action="store_true",
                    help="cfg2 with the continuous-chasing rule on (not a BASELINE.json config; the paper's simulator goal "
                         "of ~10 M updates/s is stated with its anti-chasing rules on, PAPER.md:228)")
    ap.add_argument("--skip-e2e", action="store_true", help="profiling runs: skip the host-buffer leg")
    ap.add_argument("--skip-cpu", action="store_true", help="profiling runs: skip the oracle timing")
    ap.add_argument("--profile-range", type=int, default=0, metavar="K",
                    help="profiling runs (ncu --replay-mode range): after the warm-up, "
                         "K back-to-back fused steps between cudaProfilerStart/Stop, nothing else; prints no bench line")
    args = ap.parse_args()
    if args.gpus > 1 and args.impl == "b200" and (args.workload != "cfg2" or args.profile_range):
        raise SystemExit("bench.py: --gpus > 1 is the sharded headline workload (cfg2) only; the other workloads are 1-GPU lines")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_ranks(args))
    if args.profile_range:
        run_profile_range(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.workload in ("cfg0", "cfg1"):
        run_small(args, int(args.workload[3]))
    elif args.workload == "cfg3":
        run_cfg3(args)
    elif args.workload == "cfg4":
        run_cfg4(args)
    elif args.workload == "hist":
        run_hist(args)
    elif args.workload == "search":
        run_search(args)
    elif args.workload == "infostate487":
        run_infostate(args)
    elif args.workload == "observe":
        run_observe(args)
    elif args.workload == "observe2":
        run_observe2(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
