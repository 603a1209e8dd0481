#!/usr/bin/env python
"""bench.py — env-steps/s of the fused drone-env step on N B200s (BASELINE.json metric, config 5).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5]

One "step" is one control step of the whole batch (action decode -> K substeps -> obs/reward/done/
auto-reset) = ONE kernel launch.  The timed region is R back-to-back repeats of K steps, one CUDA-event pair
per repeat; `ms_per_step` is the MEDIAN repeat (min / max / repeats beside it).  See DESIGN.md §7 for what
each JSON key means and how the roofline numbers are derived.  `--impl reference` times the float64 oracle
on the host cores (a baseline, not the target).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_08039_b200 import workloads as W  # noqa: E402
from paper_2606_08039_b200.sharding import max_over_ranks, replica_base  # noqa: E402

METRIC = "env_steps_per_sec"
UNIT = "env-steps/s"
# FP32 ALU peak: 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz (clocks.max.sm)
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# algorithmic flops per drone per control step, tallied by the oracle's counting scalar type on the
# seeded workloads (tests/test_oracle_control_env.py::test_flop_tally...)
FLOPS_PER_DRONE_STEP = {1: 3186.0, 2: 3421.1, 3: 3350.0, 4: 3893.6, 5: 3858.75}
SURVEY_FLOPS_PER_DRONE_STEP = {1: 2750.0, 2: 2960.0, 3: 2870.0, 4: 3800.0, 5: 3540.0}   # SURVEY.md 8(d) hand tally (DESIGN.md 6 reconciles the two)
REPLICAS = 4          # independent env batches stepped round-robin so the working set exceeds the 126 MB L2


VARIANTS = W.VARIANTS      # secondary workloads (`--variant`, never the default line): the overrides the parity tests run too
GRAPH_STEPS = 48          # steps per captured CUDA graph (REPLICAS batches x 12 steps, round-robin)


def algorithmic_bytes_per_drone(wl) -> float:
    """State read once + written once, actions read, outputs written; the optional planes when they are on."""
    M = wl.n_drones
    pid = wl.action_type in (W.ACT_PID, W.ACT_VEL, W.ACT_ATTITUDE)       # actions with an attitude loop read/write P4
    rd = 4 * 16 + 16 + 16 + (16 if pid else 0) + (16 if wl.action_type == W.ACT_PID else 0)   # P0-P3, target, action, P4, P5
    wr = 4 * 16 + (16 if pid else 0) + (16 if wl.action_type == W.ACT_PID else 0)
    obs = 4 * (12 + (M if wl.params.get("obs_mode", 0) == W.OBS_KIN12_ADJ else 0))
    env = (16 + 4) + (16 + 4 + 4 + 1)                                                         # per env: E0 + gstep r/w, reward, done
    extra = 0
    if any(wl.params.get("dr_alpha", [])) or wl.params.get("motor_lag_hi", 0) > 0:
        extra += 64                                                                             # R0-R3 read
    if wl.params.get("motor_lag_hi", 0) > 0:
        extra += 32                                                                             # N0 read + written
    if wl.params.get("act_latency_hi", 0) > 0:
        extra += 96                                                                             # H0-H2 read + written
    return rd + wr + obs + 4 + env / M + extra                                                # + the per-drone reward share


class ClockSampler:
    """nvidia-smi SM clock / throttle-reason samples while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.samples, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc:
            time.sleep(0.05)
            self.proc.terminate()
        mhz, mx, reasons = [], 0.0, set()
        for ts, line in self.samples:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                mx = max(mx, float(f[1]))
                if t0 <= ts <= t1 + 0.05:
                    mhz.append(float(f[0]))
                    for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
            except ValueError:
                pass
        mhz.sort()
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(mhz)}


def harness_actions(wl):
    kind = wl.actions[0]
    if kind == "hover_scale":
        return W.hover_rpm_f32(), wl.actions[1], wl.actions[2]
    if kind == "uniform":
        return 1.0, wl.actions[1], wl.actions[2]
    return None


def oracle_throughput(wl, budget_s, n_envs, min_steps=4, max_steps=10 ** 9, threads=None):
    """Time the oracle as it stands on a bounded sample of the workload: env-steps/s on `threads` host cores (default: all)."""
    import numpy as np
    from oracle import oracle as O
    cores = threads or len(os.sched_getaffinity(0))
    sample = wl.scaled(min(wl.n_envs, n_envs))
    env = O.OracleEnv(sample.n_envs, sample.n_drones, sample.physics_mode, sample.action_type, O.OracleParams(0, **sample.params), n_threads=cores)
    env.reset(sample.seed)
    ha = harness_actions(sample)
    acts = []
    for t in range(8):
        acts.append(O.gen_actions(sample.seed, t, sample.n_envs, sample.n_drones, *ha) if ha else env.targets.astype(np.float32))
    flops = env.flop_tally(acts[0]) / (sample.n_envs * sample.n_drones)
    env.step(acts[0])                                   # warm-up (thread start, page faults)
    t0 = time.perf_counter()
    steps = 0
    while steps < max_steps and (steps < min_steps or time.perf_counter() - t0 < budget_s):
        env.step(acts[steps % 8] if ha else env.targets.astype(np.float32))
        steps += 1
    dt = time.perf_counter() - t0
    return dict(value=sample.n_envs * steps / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{sample.n_envs} envs x {sample.n_drones} drones x {steps} control steps of {wl.name} (float64, {cores} threads, {dt:.1f} s)",
                flops_per_drone_step=flops, ms_per_step=1e3 * dt / steps, steps=steps)


def camera_leg(stream, hbm_peak, n_envs=16384, n_drones=4, reps=20, cpu_envs=8192):
    """Secondary measurement: mdg_render_depth, every drone's 48 x 64 depth + segmentation frame.
    16,384 envs x 4 drones = 65,536 frames = 1.0 GB of output per call (> 126 MB L2, so every call's stores reach HBM).
    Algorithmic bytes per frame: H W (4 + 1) written + the drone's 32-byte pose read."""
    import torch
    import numpy as np
    import paper_2606_08039_b200 as mdg
    with torch.cuda.stream(stream):
        env = mdg.Env(n_envs, n_drones, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, auto_reset=0, term_mode=W.TERM_NONE), stream=stream)
        env.reset(1)
        st = W.camera_scene(W.BASE_SEED + 99, n_envs, n_drones)
        env.set_state(state=st)
        depth, seg = env.render_depth()
        for _ in range(3):
            env.render_depth(depth=depth, seg=seg)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            env.render_depth(depth=depth, seg=seg)
        e1.record(stream)
        stream.synchronize()
        rgba = env.render_rgba()
        for _ in range(3):
            env.render_rgba(rgba=rgba)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        for _ in range(reps):
            env.render_rgba(rgba=rgba)
        c1.record(stream)
        stream.synchronize()
    sec = e0.elapsed_time(e1) / 1e3 / reps
    sec_rgba = c0.elapsed_time(c1) / 1e3 / reps
    frames = n_envs * n_drones
    byt = frames * (48 * 64 * 5 + 32)
    byt_rgba = frames * (48 * 64 * 4 + 32)
    out = {"workload": f"{n_envs} envs x {n_drones} drones, one 48 x 64 depth (fp32) + segmentation (u8) frame per drone, formation-circle scenes",
           "frames_per_sec": frames / sec, "us_per_call": sec * 1e6, "gpu_launches": 2 * reps,
           "rgba": {"workload": "the same scenes, one 48 x 64 x 4 uint8 colour frame per drone (mdg_render_rgba)", "frames_per_sec": frames / sec_rgba,
                    "us_per_call": sec_rgba * 1e6, "bytes_per_launch": byt_rgba, "achieved_gbs": byt_rgba / sec_rgba / 1e9,
                    "frac": byt_rgba / sec_rgba / 1e9 / hbm_peak, "kernel": "render_depth_kernel<rgba>"},
           "roofline": {"bound": "hbm", "achieved": byt / sec / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": byt / sec / 1e9 / hbm_peak,
                        "traffic": None, "kernel": "render_depth_kernel<two-pass>", "bytes_per_launch": byt,
                        "frac_of_nominal": byt / sec / 1e9 / 7700.0,
                        "peak_note": "peak = the measured COPY bandwidth (read + write stream); this kernel is a write-only stream, which can "
                                     "exceed it; frac_of_nominal is against the 7.7 TB/s HBM3e figure of B200_PROFILING.md"}}
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv"))):
            if row["config"] == "camera":
                out["roofline"]["traffic"] = float(row["traffic_bytes"])
    except Exception:
        pass
    from oracle import oracle as O
    cores = len(os.sched_getaffinity(0))
    cpu_envs = max(1, min(n_envs, cpu_envs * 16 // (n_drones * n_drones)))     # the oracle's cost per frame grows with the drones per env
    sub = st[: cpu_envs * n_drones].astype(np.float64)
    t0 = time.perf_counter()
    O.render_depth(sub, cpu_envs, n_drones, n_threads=cores)
    dt = time.perf_counter() - t0
    out["cpu_baseline"] = {"value": cpu_envs * n_drones / dt, "unit": "frames/s", "cores": cores, "kind": "oracle",
                           "sample": f"{cpu_envs} envs x {n_drones} drones of the same scenes (float64, {cores} threads, {dt:.2f} s)"}
    return out


def run_reference(args, wl, c):
    """`--impl reference`: the oracle on the host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    total = args.steps + args.warmup
    # bounded sample per step, sized from a short calibration so the whole run takes about a minute
    cal = oracle_throughput(wl, budget_s=1.0, n_envs=1024, min_steps=2)
    per_step_envs = int(max(64, min(wl.n_envs, 60.0 * cal["value"] / total)))
    res = oracle_throughput(wl, budget_s=1e9, n_envs=per_step_envs, min_steps=total, max_steps=total)
    line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_dict(wl, c, args.gpus),
            "cpu_baseline": {"value": res["value"], "unit": UNIT, "cores": res["cores"], "kind": "oracle", "sample": res["sample"]},
            "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def config_dict(wl, c, n_gpus):
    return {"workload": f"config {c} of BASELINE.json: {wl.n_envs} envs x {wl.n_drones} CF2X drones per GPU, "
                        f"physics_mode={wl.physics_mode} aero_mask={wl.params.get('aero_mask', 'from mode')}, action_type={wl.action_type}, "
                        f"240 Hz physics / 48 Hz control (5 substeps), auto-reset on"
                        + (f"; VARIANT {wl.name.split('+', 1)[1]} (secondary workload, generic kernel)" if "+" in wl.name else ""),
            "n_envs_per_gpu": wl.n_envs, "n_drones": wl.n_drones, "substeps": 5, "seed": wl.seed,
            "parallelism": f"env-sharded x{n_gpus}, no collective on the step path",
            "l2": f"{REPLICAS} independent env batches stepped round-robin (working set > 126 MB L2)"}


def capture_round_robin(torch, envs, acts, stream, n_steps, branches=False):
    """One CUDA graph of n_steps chained steps over the env batches, round-robin (caller-side capture of mdg_step_chained: a
    replayed graph chains like the stream it was captured from).  branches: each batch's steps are captured on a
    stream of their own, forked from and joined back to the capturing stream, so the graph holds one chain per batch and the
    (independent) batches step side by side - what a small batch needs to fill the device."""
    A = len(acts[0])
    g = torch.cuda.CUDAGraph()
    side = [torch.cuda.Stream() for _ in envs[1:]] if branches else []
    with torch.cuda.graph(g, stream=stream):
        cs = torch.cuda.current_stream()
        fork = torch.cuda.Event()
        fork.record(cs)
        for s_ in side:
            s_.wait_event(fork)
        for i, e in enumerate(envs):
            e.set_stream(side[i - 1] if branches and i else cs)
        for k in range(n_steps):
            envs[k % len(envs)].step_chained(acts[k % len(envs)][(k // len(envs)) % A])
        for s_ in side:
            join = torch.cuda.Event()
            join.record(s_)
            cs.wait_event(join)
    for e in envs:
        e.set_stream(stream)
    return g


def timed_repeats(torch, stream, body, repeats):
    """R back-to-back repeats of body() on `stream`, one event pair per repeat; returns the per-repeat milliseconds."""
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(repeats + 1)]
    evs[0].record(stream)
    for r in range(repeats):
        body()
        evs[r + 1].record(stream)
    stream.synchronize()
    return [evs[r].elapsed_time(evs[r + 1]) for r in range(repeats)]


def run_ours(args, wl, c):
    import torch
    import paper_2606_08039_b200 as mdg
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K, Wm = args.steps, max(args.warmup, 3)
    # the latency-bound batches (configs 1-4: at most 16,384 drones) go through one graph: no host launch rate in the number
    use_graph = args.mode == "graph" or (args.mode == "auto" and wl.n_envs * wl.n_drones < 65536)
    if use_graph:
        K = -(-K // GRAPH_STEPS) * GRAPH_STEPS                              # whole graphs
    stream = torch.cuda.Stream()
    ha = harness_actions(wl)
    A = GRAPH_STEPS // REPLICAS                            # distinct action sets per replica (12: a short period lets open-loop rotor commands pump the body rates)
    envs, acts = [], []
    with torch.cuda.stream(stream):
        for r in range(REPLICAS):
            over = dict(wl.params, env_index_base=replica_base(rank, r, REPLICAS, wl.n_envs))
            env = mdg.Env(wl.n_envs, wl.n_drones, wl.physics_mode, wl.action_type, mdg.default_params(0, **over), stream=stream)
            if args.block or args.max_blocks:
                env.set_launch(args.block, args.max_blocks)
            env.reset(wl.seed)
            envs.append(env)
            if ha:
                acts.append([env.gen_actions(wl.seed, t, *ha) for t in range(A)])
            else:
                acts.append([env.targets] * A)             # PID waypoint = the live per-episode target plane (written by the step itself, item by item)
        stream.synchronize()

        # The actions are complete before the first step is enqueued, which is mdg_step_chained's contract: consecutive steps
        # of a batch order themselves item by item, the steps of the other batches in between overlap.
        def run_stream(n):
            for k in range(n):
                envs[k % REPLICAS].step_chained(acts[k % REPLICAS][(k // REPLICAS) % A])

        branches = use_graph and args.mode == "auto"           # the latency-bound batches: one chain per batch, side by side
        graph = capture_round_robin(torch, envs, acts, stream, GRAPH_STEPS, branches=branches)

        def run_graph(n):
            with torch.cuda.stream(stream):
                for _ in range(n // GRAPH_STEPS):
                    graph.replay()

        run = run_graph if use_graph else run_stream
        run(max(Wm, GRAPH_STEPS) if use_graph else Wm)
        # One timed interval = `group` back-to-back rounds of K steps (an event pair per interval): an event between two launches
        # makes the second wait for the first as a whole, i.e. every interval pays one pipeline fill and drain; with K = 20 that
        # would be 5 % of the interval, so short K are grouped to at least 100 steps per interval (all counted, all reported).
        group = max(1, -(-100 // K))
        body = lambda: [run(K) for _ in range(group)]
        # size the block of repeats: at least 7, and long enough (0.6 s) for the clock sampler to see the GPU under this load
        pre = timed_repeats(torch, stream, body, 3)
        est = sorted(pre)[1] / 1e3
        R = int(max(7, min(args.max_repeats, 0.6 / max(est, 1e-6))))
        if dist:
            rt = torch.tensor([R], device="cuda")
            dist.all_reduce(rt, op=dist.ReduceOp.MAX)
            R = int(rt.item())
            dist.barrier()
        torch.cuda.synchronize()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
            time.sleep(0.1)
        l0 = sum(e.launch_count for e in envs)
        t_wall0 = time.time()
        per_repeat = [x / group for x in timed_repeats(torch, stream, body, R)]      # ms per K steps
        torch.cuda.synchronize()
        t_wall1 = time.time()
        if dist:
            dist.barrier()
        launches = (R * K * group) if use_graph else (sum(e.launch_count for e in envs) - l0)
        clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
        srt = sorted(per_repeat)
        ms, ms_min, ms_max = srt[len(srt) // 2], srt[0], srt[-1]
        ms, ms_min, ms_max = (max_over_ranks(x, dist, "cuda") for x in (ms, ms_min, ms_max))
        # the other launch path beside the headline one: K steps as replays of one captured graph / as a stream of launches
        other = run_stream if use_graph else run_graph
        Ko = -(-K // GRAPH_STEPS) * GRAPH_STEPS
        other(Ko)
        alt = sorted(timed_repeats(torch, stream, lambda: other(Ko), 7))[3]
        alt = max_over_ranks(alt, dist, "cuda")
        one_chain = None                                       # the same graph with all batches on ONE chain, for comparison
        if branches:
            g1 = capture_round_robin(torch, envs, acts, stream, GRAPH_STEPS)

            def run_g1(n):
                with torch.cuda.stream(stream):
                    for _ in range(n // GRAPH_STEPS):
                        g1.replay()
            run_g1(Ko)
            one_chain = max_over_ranks(sorted(timed_repeats(torch, stream, lambda: run_g1(Ko), 7))[3], dist, "cuda")
        # ---- end to end through the C ABI with host buffers (pinned): H2D actions, step, D2H obs/reward/done, every step.
        # (a) one batch, the synchronous call (mdg_step_host); (b) two batches double-buffered on two streams
        # (mdg_step_host_async / mdg_wait): the host consumes batch A's results while batch B is in flight, so one batch's
        # D2H overlaps the other's H2D and step (PCIe is full duplex).  (b) is the headline e2e; (a) is reported beside it.
        env = envs[0]
        D = wl.n_envs * wl.n_drones
        a_host = [a.cpu().pin_memory() for a in acts[0]]
        Ke = max(4, min(K, args.e2e_steps)) // 2 * 2

        def host_bufs():
            return (torch.empty((wl.n_envs, env.obs_dim), dtype=torch.float32).pin_memory(),
                    torch.empty(wl.n_envs, dtype=torch.float32).pin_memory(), torch.empty(wl.n_envs, dtype=torch.uint8).pin_memory())
        bufs = [host_bufs(), host_bufs()]
        for k in range(3):
            env.step_host(a_host[k % A], *bufs[0])
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(Ke):
            env.step_host(a_host[k % A], *bufs[0])
        e1.record(stream)
        torch.cuda.synchronize()
        ms_e2e_single = e0.elapsed_time(e1)
        # (b): envs[0] stays on `stream`, envs[1] moves to a second stream for this leg
        stream_b = torch.cuda.Stream()
        pair, streams = [envs[0], envs[1]], [stream, stream_b]
        envs[1].set_stream(stream_b)
        a_host_b = [a.cpu().pin_memory() for a in acts[1]]
        ah = [a_host, a_host_b]
        for k in range(4):
            pair[k % 2].step_host(ah[k % 2][(k // 2) % A], *bufs[k % 2])
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        e0, e1, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event()
        e0.record(stream)
        stream_b.wait_event(e0)                               # batch B's work starts inside the timed region
        pair[0].step_host(ah[0][0], *bufs[0], asynchronous=True)
        for k in range(1, Ke):
            pair[k % 2].step_host(ah[k % 2][(k // 2) % A], *bufs[k % 2], asynchronous=True)
            pair[(k - 1) % 2].wait()                           # the other batch's results are on the host now (a policy would read them here)
        pair[(Ke - 1) % 2].wait()
        eb.record(stream_b)
        stream.wait_event(eb)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_e2e = e0.elapsed_time(e1)
        envs[1].set_stream(stream)
        if dist:
            tt = torch.tensor([ms_e2e, ms_e2e_single], device="cuda")
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            ms_e2e, ms_e2e_single = float(tt[0].item()), float(tt[1].item())
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return
    sec = ms / 1e3
    value = world * wl.n_envs * K / sec
    per_launch_s = sec / K
    drones = wl.n_envs * wl.n_drones
    cpu = oracle_throughput(wl, budget_s=args.cpu_budget, n_envs=16384) if world == 1 and not args.no_cpu else None
    cpu1 = oracle_throughput(wl, budget_s=args.cpu_budget / 3, n_envs=2048, threads=1) if cpu else None
    fpd = cpu["flops_per_drone_step"] if cpu else FLOPS_PER_DRONE_STEP[c]
    flops = fpd * drones
    bytes_alg = algorithmic_bytes_per_drone(wl) * drones
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    try:
        ffma_tf = mdg.measure_fp32_peak(stream)              # FFMA microbenchmark on this GPU, this run
    except Exception:
        ffma_tf = None
    achieved_tf = flops / per_launch_s / 1e12
    t_alu, t_hbm = flops / (ALU_PEAK_TFLOPS * 1e12), bytes_alg / (hbm_peak * 1e9)
    traffic = None                                         # dram read + write bytes per launch, one ncu --set full capture
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv"))):
            if row["config"] == (f"c{c}+{args.variant}" if args.variant else f"c{c}"):
                traffic = float(row["traffic_bytes"])
    except Exception:
        pass
    traffic_timed = None                                   # the same, summed over four consecutive launches of the four batches / 4
    try:
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv"))):
            if row["config"] == (f"c{c}+{args.variant}_timed" if args.variant else f"c{c}_timed"):
                traffic_timed = float(row["traffic_bytes"])
    except Exception:
        pass
    cfg = config_dict(wl, c, world)
    cfg["launch_path"] = ((f"replays of one CUDA graph of {GRAPH_STEPS} chained steps (caller-side capture of mdg_step_chained)"
                           + (f", one chain per batch on {REPLICAS} concurrent branches" if branches else "")) if use_graph
                          else "a stream of mdg_step_chained launches (actions pre-generated and resident: its contract)")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": ms / K,
            "repeats": R, "steps_per_timed_interval": K * group, "ms_per_step_min": ms_min / K, "ms_per_step_max": ms_max / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cfg,
            ("stream" if use_graph else "graph"): {"ms_per_step": alt / Ko, "steps_per_graph": GRAPH_STEPS, "steps": Ko, "repeats": 7,
                                                     "value": world * wl.n_envs * Ko / (alt / 1e3)},
            **({"graph_one_chain": {"ms_per_step": one_chain / Ko, "steps_per_graph": GRAPH_STEPS, "steps": Ko, "repeats": 7}} if one_chain else {}),
            "drone_substeps_per_sec": value * wl.n_drones * 5,
            "roofline": {"bound": "alu", "achieved": achieved_tf, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved_tf / ALU_PEAK_TFLOPS,
                         "traffic": traffic, "traffic_timed": traffic_timed, "kernel": envs[0].kernel_name,
                         "frac_survey_tally": SURVEY_FLOPS_PER_DRONE_STEP[c] * drones / per_launch_s / 1e12 / ALU_PEAK_TFLOPS, "us_per_launch": per_launch_s * 1e6,
                         "flops_per_launch": flops, "bytes_per_launch": bytes_alg,
                         "peak_note": "FP32 ALU peak derived: 148 SMs x 128 lanes x 2 x 1.965 GHz (DESIGN.md §6)",
                         "ffma_measured_tflops": ffma_tf, "frac_of_ffma_measured": (achieved_tf / ffma_tf) if ffma_tf else None,
                         "hbm": {"achieved_gbs": bytes_alg / per_launch_s / 1e9, "peak_gbs": hbm_peak,
                                 "peak_source": "MEASURED_PEAKS.json (measured)" if peaks else "fallback of B200_PROFILING.md",
                                 "frac": bytes_alg / per_launch_s / 1e9 / hbm_peak},
                         "t_roof_us": max(t_alu, t_hbm) * 1e6, "frac_of_binding_roof": max(t_alu, t_hbm) / per_launch_s},
            "e2e": {"value": world * wl.n_envs * Ke / (ms_e2e / 1e3), "unit": UNIT, "h2d_bytes_per_step": drones * 16,
                    "d2h_bytes_per_step": wl.n_envs * env.obs_dim * 4 + wl.n_envs * 5, "steps": Ke, "ms_per_step": ms_e2e / Ke,
                    "mode": "two env batches double-buffered on two streams (mdg_step_host_async / mdg_wait), pinned host buffers",
                    "single_batch_value": world * wl.n_envs * Ke / (ms_e2e_single / 1e3), "single_batch_ms_per_step": ms_e2e_single / Ke},
            "gpu_launches": launches, "clocks": clocks}
    if cpu:
        line["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
        line["cpu_baseline"]["single_thread_value"] = cpu1["value"]
        line["cpu_baseline"]["single_thread_sample"] = cpu1["sample"]
    if world == 1 and not args.no_camera:
        del envs, acts
        torch.cuda.empty_cache()
        line["camera"] = camera_leg(stream, hbm_peak, n_envs=65536 // args.camera_drones, n_drones=args.camera_drones)
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config 1..5 (5 = 65,536 envs x 4 drones, the metric's config)")
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--max-blocks", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--mode", default="auto", choices=["auto", "stream", "graph"],
                    help="launch path of the timed region: a stream of mdg_step_chained calls, or replays of one captured CUDA graph "
                         "(auto: stream for config 5, graph for the latency-bound configs 1-4); the other one is reported beside it")
    ap.add_argument("--max-repeats", type=int, default=2000)
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-camera", action="store_true", help="skip the secondary onboard-camera measurement")
    ap.add_argument("--camera-drones", type=int, default=4, help="drones per env of the camera measurement (65,536 cameras in all)")
    ap.add_argument("--variant", default="", choices=["", "dyn", "table4", "noise", "paper_mjx"], help="secondary workload on the chosen config (see VARIANTS)")
    args = ap.parse_args()
    wl = W.config(args.config)
    if args.variant:
        if args.no_cpu:
            raise SystemExit("--variant needs the oracle leg: its flop tally is the roofline numerator")
        if args.variant == "paper_mjx":
            # the workload of the paper's own MJX back end (hover, rigid body only, normalised rotor commands,
            # PAPER.md:300), at 2^20 envs ("the only practical limit is GPU memory") instead of its default 4,096
            args.config = 1
            base = W.config(1)
            wl = W.Workload("c1", 1 << 20, 1, W.PHYS_MJC, W.ACT_RPM_NORM, dict(base.params), ("uniform", -0.05, 0.06), 1000, base.seed)
        else:
            wl.params.update(VARIANTS[args.variant])
        wl.name += "+" + args.variant
    if args.impl == "reference":
        run_reference(args, wl, args.config)
    else:
        run_ours(args, wl, args.config)


if __name__ == "__main__":
    main()
