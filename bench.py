#!/usr/bin/env python
"""bench.py -- BR-MPPI throughput on synthetic parking scenes (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2]

A "step" is one control-step solve of the whole hot path (DESIGN.md §2 rows a1-a8: n_iter x
{noise, perturb+clamp, rollout, barrier-rate + costs, online-softmax reduction, update}) on one
synthetic scene.  Default workload: BASELINE.json configs[2] (K=16384, T=80, 8 obstacles of which
3 move, 3 iterations per control step) -- the config the north star's ">= 50 % at K >= 16384" and
"control rate at the 8-obstacle config" are quoted on.

One JSON line on stdout (rank 0).  `value` = sample-steps/s with inputs resident in HBM, device
time from CUDA events on the solver's stream, L2 flushed between steps; `e2e` = the same metric
through the C ABI with host buffers (set_state/goal/obstacles from pinned host memory, solve,
get_controls back to the host) on the host clock.  `roofline` is for the rollout kernel
(DESIGN.md §6); `cpu_baseline` is the fp64 oracle on this box's host cores (a reported baseline,
not the target).  --impl reference times that oracle alone.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import scenes  # noqa: E402

N_SMS = 148
ISSUE_PER_CLK_PER_SM = 128          # thread-instructions per clock per SM (4 schedulers x 32 lanes)
SM_MAX_MHZ_FALLBACK = 1965.0
METRIC = "brmppi_sample_steps_per_s"
UNIT = "sample-steps/s"


def workload(name, rank=0):
    """Scene + params of a named workload; rank r uses scene seed r (independent replicas)."""
    if name == "cfg0":
        sc = scenes.scene_cfg0(rank)
    elif name == "cfg1":
        sc = scenes.scene_cfg1(rank)
    elif name == "cfg2":
        sc = scenes.scene_cfg2(rank)
    elif name == "cfg2se":
        sc = scenes.scene_cfg2_superellipse(rank)
    elif name == "cfg3":
        sc = scenes.scene_cfg3(rank)
    elif name == "cfg2proj":      # CFG2 solved by BR-MPPI proper: projection (9)-(12) inside the rollout
        sc = scenes.scene_cfg2(rank)
    elif name == "paperproj":     # the paper's own size: 5000 rollouts x H = 120 (T_s = 0.04 s) x 8 obstacles
        sc = scenes.scene_cfg2(rank)
        sc.params = sc.params.with_(K=5000, T=120, dt=0.04, n_iter=1)
    elif name == "cfg2mpcc":      # CFG2's size on the paper's own model and cost: 7 states, predictor (17), cost (13)
        sc = scenes.scene_mpcc(rank, K=16384, T=80, dt=0.05, n_obs=8, M=24)
        sc.params = sc.params.with_(n_iter=3)
    elif name == "papermpcc":     # the paper's own size on the paper's own model
        sc = scenes.scene_mpcc(rank, K=5000, T=120, dt=0.04, n_obs=8, M=24)
    else:
        raise SystemExit(f"unknown workload {name}")
    return sc, sc.params


PROJECTED = ("cfg2proj", "paperproj")
MPCC = ("cfg2mpcc", "papermpcc")
LONG_STEPS = PROJECTED + MPCC                 # workloads whose control step takes 0.1 ms or more: fewer timed steps


def solver_flags(B, name, no_cull=False):
    return ((B.FLAG_PROJECTED if name in PROJECTED else 0) | (B.FLAG_MPCC if name in MPCC else 0) |
            (B.FLAG_NO_CULL if no_cull else 0))


def oracle_solve(O, name, ps, n0, sc, U, n_threads):
    if name in MPCC:
        return O.solve7(ps, sc.coef, sc.dpsi, n0, sc.x0, sc.psi0, sc.obstacles, U, n_threads=n_threads)
    if name in PROJECTED:
        return O.solve_projected(ps, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=n_threads)
    return O.solve(ps, n0, sc.x0, sc.goal, sc.obstacles, U, n_threads=n_threads, superellipses=sc.superellipses)


def projected_instr_per_sample_step(n_obs, n_discs):
    """issue slots of one projected sample-step.  150 fixed (control noise, perturb + clamp,
    model step, tracking cost); 64 per Philox block of auxiliary-input normals (one per four obstacles);
    16 + 10 D per row of (9) (obstacle position, D disc barriers, closest disc, gradient, L_g h, L_f h, b);
    the projection (12): y, r, S = A M^-1 A^T from its rank-2-plus-diagonal form, Cholesky, two triangular
    solves, z*, alpha update."""
    N = n_obs
    chol = N * (N - 1) // 2 + sum((N - 1 - c) * (c + 1) for c in range(N)) + 3 * N
    proj = 14 + 4 * N + N * (N + 1) + chol + (N * (N - 1) + 2 * N) + (4 * N + 2) + 3 * N
    return 150 + 64 * ((N + 3) // 4) + N * (16 + 10 * n_discs) + proj


def mpcc_instr_per_sample_step(n_obs, n_discs):
    """issue slots of one sample-step of the paper's own model and cost, with the predictor folded
    into one quadratic form per (obstacle, disc) (rollout_mpcc.cuh: mpcc_hinge).  Fixed 203: noise, perturb and clamp
    60 (as on the penalty path); sin / cos of the two headings, tan and sec^2 of delta 11; sin / cos of the hitch
    angle 4; step-unit scaling 3; W1, W2 and their time derivatives 20; the six vectors every disc's velocity and
    acceleration are affine in 24; Euler step (6) 12; path segment and four cubics 19; tracking errors (14), (15),
    heading wraps, nu 26; progress, effort, hitch hinge, psi update, accumulate, loop 24.  Per disc 12: centre,
    velocity, 2 v + a.  Per obstacle 2 (position); per (obstacle, disc) 16: differences 4, obstacle-velocity
    correction 2, d.(2e + a) + |e|^2 4, |d|^2 2, alpha |d|^2 1, alpha - q / rho^2 1, max and accumulate 2."""
    return 203 + 12 * n_discs + n_obs * (2 + 16 * n_discs)


def algorithmic_instr_per_sample_step(n_obs, n_discs, superellipses=None, philox_per_step=1.0):
    """SURVEY.md §8(d) / DESIGN.md §6: issue slots the method itself needs per sample-step.
    Discs: 8 per (obstacle, disc).  Super-ellipses (eq. 16): 2 differences, 4 for the rotation and
    scaling, 4 (e = 4) or 2 (e = 2) for the powers and their sum, rate argument, max, accumulate.
    philox_per_step: the survey's 121 charges one Philox block (40 slots) per step; reading 6 draws one block
    per PAIR of steps (0.5 -> 101 fixed slots)."""
    n = 121 - int(round(40 * (1.0 - philox_per_step))) + 8 * n_obs * n_discs
    if superellipses is not None:
        for row in superellipses:
            n += (13 if int(round(row[7])) == 4 else 11) * n_discs
    return n


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return json.load(open(path))
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, val in zip(names, r[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_throughput(sc, p, seconds_target, n_threads, k_sample, name="cfg2"):
    """Time the oracle, as it stands, on a bounded sample (k_sample of the K samples, all T steps,
    all n_iter iterations).  Returns (sample-steps/s, seconds, description)."""
    from oracle import oracle as O
    O.lib()
    ps = p.with_(K=k_sample)
    U = np.zeros((p.T, 2))
    t0 = time.perf_counter()
    reps = 0
    while True:
        oracle_solve(O, name, ps, reps * p.n_iter, sc, U, n_threads)
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= seconds_target or reps >= 50:
            break
    work = reps * k_sample * p.T * p.n_iter
    return work / dt, dt, f"{reps} x ({k_sample} of {p.K} samples x T={p.T} x {p.n_iter} iterations), {n_threads} thread(s)"


def dist_setup(n_gpus):
    """(rank, world, local_rank, dist-or-None).  Under torchrun the env carries the rendezvous."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world <= 1:
        return 0, 1, 0, None
    import torch.distributed as dist
    backend = os.environ.get("BRMPPI_DIST_BACKEND", "nccl")
    dist.init_process_group(backend=backend)
    return dist.get_rank(), dist.get_world_size(), int(os.environ.get("LOCAL_RANK", "0")), dist


def max_over_ranks(seconds, dist, device):
    """Every rank's device time -> the slowest rank's (the job is as slow as its slowest GPU)."""
    if dist is None:
        return float(seconds)
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(work_per_rank, world, seconds_max):
    """Replicas: every rank processes `work_per_rank` units in at most `seconds_max`."""
    return world * work_per_rank / seconds_max


def run_reference(args):
    """The reference arm of this tier is the oracle, timed as it stands on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return                                      # rank 0 alone runs it; the others exit 0
    sc, p = workload(args.workload)
    cores = os.cpu_count() or 1
    k_sample = min(p.K, 1024)
    from oracle import oracle as O
    O.lib()
    ps = p.with_(K=k_sample)
    U = np.zeros((p.T, 2))
    for w in range(args.warmup):
        oracle_solve(O, args.workload, ps, w, sc, U, cores)
    t0 = time.perf_counter()
    for s in range(args.steps):
        oracle_solve(O, args.workload, ps, s, sc, U, cores)
    dt = time.perf_counter() - t0
    value = args.steps * k_sample * p.T * p.n_iter / dt
    sample = f"each step = {k_sample} of {p.K} samples x T={p.T} x {p.n_iter} iterations, {cores} threads"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, sc, p, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_config(name, sc, p, n_scenes_total):
    label = {"cfg2se": "BASELINE.json configs[2] with the paper's super-ellipse obstacles, eq. (16) (cfg2se)",
             "cfg2proj": "BASELINE.json configs[2] solved by BR-MPPI proper: projection (9)-(12) inside the rollout (cfg2proj)",
             "paperproj": "the paper's size, 5000 rollouts x H = 120 x 8 obstacles (PAPER.md:243), projected rollout of the reduced model (paperproj)",
             "cfg2mpcc": "BASELINE.json configs[2]'s size on the paper's own 7-state model, predictor (17) and contouring cost (13) (cfg2mpcc)",
             "papermpcc": "the paper's size, 5000 rollouts x H = 120 x 8 obstacles (PAPER.md:243), on the paper's own 7-state model and contouring cost (papermpcc)",
             }.get(name, f"BASELINE.json configs[{name[-1]}] ({name})")
    return {"workload": label, "K": p.K, "T": p.T,
            "n_obstacles": int(len(sc.obstacles)),
            "n_superellipses": 0 if getattr(sc, "superellipses", None) is None else int(len(sc.superellipses)),
            "n_moving": int(np.count_nonzero(np.abs(sc.obstacles[:, 3:5]).sum(axis=1))) if len(sc.obstacles) else 0,
            "n_discs": len(p.discs), "n_iter": p.n_iter, "dt": p.dt, "scenes_total": n_scenes_total,
            "l2": "flushed between timed steps (256 MiB write); per-step CUDA-event pairs",
            "parallelism": "independent replicas, one scene per GPU, no collective on the data path"}


def measure(B, torch, name, rank, steps, warmup, dist, dev, local_rank, closed_loop_steps, with_clocks):
    """One workload on this rank: device-resident throughput (CUDA events on the solver's stream, L2 flushed
    between steps), end to end through the C ABI with pinned host buffers, closed-loop brmppi_step latency,
    kernel times by CUDA events (with and without culling)."""
    sc, p = workload(name, rank)
    n_obs = len(sc.obstacles)
    se = getattr(sc, "superellipses", None)
    n_se = 0 if se is None else len(se)
    n_seg = sc.coef.shape[0] if name in MPCC else 1
    solver = B.Solver(p, 1, max(n_obs, 1), solver_flags(B, name), device=dev, max_superellipses=n_se,
                      max_path_segments=n_seg)
    solver.set_scene(sc)
    stream = solver.stream
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(warmup, 3)):
        solver.solve()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    launches0 = solver.launch_count()
    sampler = ClockSampler(local_rank) if with_clocks else None
    if sampler:
        sampler.start()
    t_wall0 = time.perf_counter()
    for a, b in ev:
        with torch.cuda.stream(stream):
            flush.fill_(1)                                   # L2 flush, outside the event pair
        a.record(stream)
        solver.solve()
        b.record(stream)
    barrier()
    wall_s = time.perf_counter() - t_wall0
    launches = solver.launch_count() - launches0
    dev_s = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    dev_s_max = max_over_ranks(dev_s, dist, dev)

    # ---- end to end through the C ABI with host buffers (pinned), host clock
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory().numpy()
    hx, ho = pin(sc.x0), pin(sc.obstacles)
    hg = pin(sc.coef) if name in MPCC else pin(sc.goal)
    hs = None if n_se == 0 else se

    def set_inputs():
        if name in MPCC:
            solver.set_reference_path(hg, sc.dpsi); solver.set_state7(hx, sc.psi0); solver.set_obstacles(ho)
            return
        solver.set_inputs(hx, hg, ho)                        # state, goal, obstacles: one call, one copy
        if hs is not None:
            solver.set_superellipses(hs)
    U_host = np.empty((1, p.T, 2), dtype=np.float32)
    one_call = name not in MPCC and hs is None               # brmppi_solve_host: inputs, solve, result in ONE call
    def e2e_step():
        if one_call:                                         # one graph launch: input copy node, kernels; T*2 floats
            solver.solve_host(hx, hg, ho, U_host)            # back, written by the last update into page-locked host
        else:                                                # memory (no copy node); synchronises
            set_inputs()
            solver.solve_get_controls(U_host)
    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        e2e_step()
    barrier()
    e2e_s_max = max_over_ranks(time.perf_counter() - t0, dist, dev)
    # brmppi_set_inputs copies the padded input span of the workspace in one piece: state, goal and the obstacle
    # count in 256-byte slots, then n_obs obstacles of 20 bytes (196 payload bytes at 8 obstacles)
    h2d = 3 * 256 + 20 * n_obs + (32 * n_se + 4 if n_se else 0)
    if name in MPCC:                                         # state and psi, path table with M and dpsi, obstacles
        h2d = 32 + (64 * n_seg + 8) + 20 * n_obs + 4
    d2h = 8 * p.T

    # ---- closed-loop control rate (CUDA-graph replay of solve + plant step + shift)
    lat = []
    for i in range(20 + closed_loop_steps):
        t1 = time.perf_counter()
        solver.step()
        if i >= 20:
            lat.append(time.perf_counter() - t1)
    clocks = sampler.stop() if sampler else None             # sampled across all three timed regions
    lat.sort()
    p50, p99 = lat[len(lat) // 2], lat[min(len(lat) - 1, int(0.99 * len(lat)))]

    # ---- kernel times (rank 0): device time per launch from CUDA events on the solver's stream
    roof = None
    if rank == 0:
        solver.set_scene(sc)
        solver.set_nominal(None)
        ms_roll, ms_upd = solver.time_kernels(50)
        ms_nocull = None
        if name not in PROJECTED:                            # the same launch with every (obstacle, disc, step) evaluated
            s2 = B.Solver(p, 1, max(n_obs, 1), solver_flags(B, name, no_cull=True), device=dev, max_superellipses=n_se,
                          max_path_segments=n_seg)
            s2.set_scene(sc)
            for _ in range(3):
                s2.solve()
            s2.set_scene(sc); s2.set_nominal(None)
            ms_nocull = s2.time_kernels(50)[0]
            s2.close()
        mp = measured_peaks()
        sm_max = float(mp.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK))
        peak = N_SMS * ISSUE_PER_CLK_PER_SM * sm_max * 1e6 / 1e9
        if name in PROJECTED:
            instr = projected_instr_per_sample_step(n_obs, len(p.discs))
            instr_pair = instr
        elif name in MPCC:
            instr = mpcc_instr_per_sample_step(n_obs, len(p.discs))
            instr_pair = instr - 20
        else:
            instr = algorithmic_instr_per_sample_step(n_obs, len(p.discs), se)
            instr_pair = algorithmic_instr_per_sample_step(n_obs, len(p.discs), se, philox_per_step=0.5)
        achieved = p.K * p.T * instr / (ms_roll * 1e-3) / 1e9          # G thread-instr / s
        traffic, traffic_source = dram_traffic_from_profile()
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Ginstr/s (thread-instructions)",
                "frac": achieved / peak, "traffic": traffic if name == "cfg2" else None,
                "traffic_source": traffic_source if name == "cfg2" else None,
                "kernel": "rollout_projected" if name in PROJECTED else "rollout_mpcc_cta" if name in MPCC else "rollout_cta",
                "kernel_ms": ms_roll, "update_kernel_ms": ms_upd,
                "kernel_share_of_step": ms_roll * p.n_iter / (dev_s / steps * 1e3),
                "algorithmic_instr_per_sample_step": instr,
                "frac_with_one_philox_block_per_step_pair": p.K * p.T * instr_pair / (ms_roll * 1e-3) / 1e9 / peak,
                "algorithmic_instr_per_sample_step_pair_blocks": instr_pair,
                "kernel_ms_no_cull": ms_nocull,
                "frac_no_cull": None if ms_nocull is None else p.K * p.T * instr / (ms_nocull * 1e-3) / 1e9 / peak,
                "static_obstacles": None if name not in MPCC else "obstacles at rest take a 10-instruction form of the "
                           "predictor hinge (dropped terms are exact zeros); frac counts the general 16 per (obstacle, "
                           "disc) for all of them, as useful work (DESIGN.md 9.2)",
                "culling": None if ms_nocull is None else "exact (bit-identical results, DESIGN.md 6.5): frac counts "
                           "every (obstacle, disc, step) the method defines as useful work; frac_no_cull is the same "
                           "launch with all of them executed (BRMPPI_FLAG_NO_CULL)",
                "peak_basis": f"{N_SMS} SMs x {ISSUE_PER_CLK_PER_SM} thread-instr/clk/SM x {sm_max:.0f} MHz "
                              f"({'MEASURED_PEAKS.json sm_max_mhz' if 'sm_max_mhz' in mp else 'fallback clock'}); "
                              "issue rate confirmed by brmppi_measure_peaks (DESIGN.md §6)"}
    solver.close()
    del flush
    return dict(sc=sc, p=p, dev_s=dev_s, dev_s_max=dev_s_max, e2e_s_max=e2e_s_max, h2d=h2d, d2h=d2h, p50=p50, p99=p99,
                launches=int(launches), clocks=clocks, roof=roof, wall_s=wall_s, steps=steps)


def record(name, m, world):
    """Compact record of a secondary workload for the `others` key of the JSON line."""
    p, steps = m["p"], m["steps"]
    work = steps * p.K * p.T * p.n_iter
    r = m["roof"] or {}
    return {"workload": name, "K": p.K, "T": p.T, "n_obstacles": int(len(m["sc"].obstacles)), "n_iter": p.n_iter, "steps": steps,
            "value": world * work / m["dev_s_max"], "unit": UNIT, "ms_per_step": m["dev_s_max"] / steps * 1e3,
            "e2e_value": world * work / m["e2e_s_max"],
            "closed_loop_p50_ms": m["p50"] * 1e3, "closed_loop_p99_ms": m["p99"] * 1e3, "closed_loop_hz": 1.0 / m["p50"],
            "kernel": r.get("kernel"), "kernel_ms": r.get("kernel_ms"), "update_kernel_ms": r.get("update_kernel_ms"),
            "frac": r.get("frac"), "kernel_ms_no_cull": r.get("kernel_ms_no_cull"), "frac_no_cull": r.get("frac_no_cull"),
            "algorithmic_instr_per_sample_step": r.get("algorithmic_instr_per_sample_step"), "gpu_launches": m["launches"]}


def batch64_record(B):
    """BASELINE.json configs[4]'s batched launch: 64 scenes x K = 16384, T = 80, 8 obstacles in one launch."""
    batch = scenes.scene_batch(64, 16384, 80)
    p = batch[0].params.with_(seed=0)
    s = B.Solver(p, 64, 8, 0)
    for i, sc in enumerate(batch):
        s.set_scene(sc, i)
    for _ in range(3):
        s.solve()
    s.synchronize()
    ms_roll, ms_upd = s.time_kernels(10)
    s.close()
    work = 64 * p.K * p.T
    instr = algorithmic_instr_per_sample_step(8, len(p.discs))
    peak = N_SMS * ISSUE_PER_CLK_PER_SM * float(measured_peaks().get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6
    return {"workload": "batch64", "n_scenes": 64, "K": p.K, "T": p.T, "n_obstacles": 8, "kernel_ms": ms_roll,
            "update_kernel_ms": ms_upd, "value": work / ((ms_roll + ms_upd) * 1e-3), "unit": UNIT,
            "frac": work * instr / (ms_roll * 1e-3) / peak}


def run_ours(args):
    import torch
    from paper_2508_05773_b200 import brmppi as B

    rank, world, local_rank, dist = dist_setup(args.gpus)
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(dev)
    m = measure(B, torch, args.workload, rank, args.steps, args.warmup, dist, dev, local_rank,
                min(args.steps, 200), with_clocks=(rank == 0))
    if rank != 0:
        return
    sc, p = m["sc"], m["p"]
    work_per_rank = args.steps * p.K * p.T * p.n_iter
    # the other BASELINE.json configs, the 64-scene batch and the projected rollout: N = 1 only, shorter runs
    others = []
    if world == 1 and not args.no_others:
        for name in ("cfg0", "cfg1", "cfg2", "cfg3", "cfg2se", "cfg2proj", "paperproj", "cfg2mpcc", "papermpcc"):
            if name != args.workload:
                steps_o = 20 if name in LONG_STEPS else 50
                others.append(record(name, measure(B, torch, name, 0, steps_o, 5, None, dev, local_rank, 100, False), 1))
        others.append(batch64_record(B))
    cores = os.cpu_count() or 1
    v1, s1, d1 = oracle_throughput(sc, p, 6.0, 1, min(p.K, 2048), args.workload)
    vn, sn, dn = oracle_throughput(sc, p, 8.0, cores, min(p.K, 8192), args.workload)
    cpu = {"value": vn, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": dn,
           "value_1core": v1, "sample_1core": d1}
    dev_s_max, e2e_s_max = m["dev_s_max"], m["e2e_s_max"]
    line = {
        "metric": METRIC, "value": whole_job_value(work_per_rank, world, dev_s_max), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": dev_s_max / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": workload_config(args.workload, sc, p, world),
        "solves_per_s": world * args.steps * p.n_iter / dev_s_max,
        "control_steps_per_s": world * args.steps / dev_s_max,
        "e2e": {"value": whole_job_value(work_per_rank, world, e2e_s_max), "unit": UNIT, "h2d_bytes_per_step": m["h2d"],
                "d2h_bytes_per_step": m["d2h"], "control_steps_per_s": world * args.steps / e2e_s_max},
        "closed_loop": {"p50_ms": m["p50"] * 1e3, "p99_ms": m["p99"] * 1e3, "hz": 1.0 / m["p50"],
                        "what": "brmppi_step: graph replay of solve + plant step + shift, host wall clock"},
        "gpu_launches": m["launches"], "clocks": m["clocks"], "roofline": m["roof"], "cpu_baseline": cpu,
        "wall_s_timed_region": m["wall_s"], "others": others,
        "paper_context": "paper: 9.9 ms per MPPI step, >100 Hz, 5000 rollouts x H=120, 8 obstacles, JAX on an unnamed GPU (PAPER.md:5,243) -- full formulation (7-state model, contouring cost), context only; the `papermpcc` record under `others` is the same size on the same model and cost family (7 states, predictor (17), contouring cost; penalty form of the barrier-rate condition), `paperproj` the same size solved by the projected rollout of the reduced model",
    }
    print(json.dumps(line))


def run_sharded(args):
    """K-sharded solve: the K samples of ONE solve split over the ranks, one 8 + 2T-float record
    per rank and iteration all-gathered over NCCL.  Strong scaling: total work is fixed as N grows."""
    import torch
    from paper_2508_05773_b200 import brmppi as B
    from paper_2508_05773_b200 import sharded
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29655")
        os.environ.setdefault("RANK", "0"); os.environ.setdefault("WORLD_SIZE", "1")
        dist.init_process_group(backend=os.environ.get("BRMPPI_DIST_BACKEND", "nccl"))
    rank, world = dist.get_rank(), dist.get_world_size()
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(dev)
    sc, p = workload(args.workload, 0)                       # every rank solves the SAME scene
    s = sharded.ShardedSolver(B, p, dist, 1, max(len(sc.obstacles), 1), solver_flags(B, args.workload), device=dev)
    s.set_scene(sc)
    for _ in range(max(args.warmup, 3)):
        s.solve()
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(s.solver.stream)
    for _ in range(args.steps):
        s.solve()
    b.record(s.solver.stream)
    torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()
    dev_s = max_over_ranks(a.elapsed_time(b) * 1e-3, dist, dev)
    U = s.get_controls()
    s.close()
    if rank == 0:
        work = args.steps * p.K * p.T * p.n_iter
        print(json.dumps({"metric": METRIC, "value": work / dev_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": max(args.warmup, 3), "ms_per_step": dev_s / args.steps * 1e3, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": dict(workload_config(args.workload, sc, p, 1),
                                         parallelism=f"K sharded over {world} rank(s): {p.K // world} samples per rank, one "
                                                     f"{4 * (8 + 2 * p.T)}-byte record per rank and iteration all-gathered (NCCL)"),
                          "gpu_launches": int(args.steps * p.n_iter * 3), "U0": [float(x) for x in U[0]]}))
    dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without a torchrun environment: start the N ranks here (one process per GPU)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def dram_traffic_from_profile(name="r2_rollout_cta_dram.csv"):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, where it comes from):
    NOT measured in this run -- read from the committed ncu capture profiles/<name> (header line, then bytes)."""
    try:
        rows = open(os.path.join(ROOT, "profiles", name)).read().strip().splitlines()
        return float(rows[-1].split(",")[-1]), f"profiles/{name} (committed ncu --set full capture, not this run)"
    except Exception:
        return None, None


def run_phases(args):
    """In-kernel phase times of one rollout launch (BRMPPI_FLAG_PHASE_TIMING), one JSON line."""
    import torch  # noqa: F401
    from paper_2508_05773_b200 import brmppi as B
    sc, p = workload(args.workload)
    n_se = 0 if sc.superellipses is None else len(sc.superellipses)
    s = B.Solver(p.with_(n_iter=1), 1, max(len(sc.obstacles), 1), B.FLAG_PHASE_TIMING | (B.FLAG_NO_CULL if args.no_cull else 0),
                 max_superellipses=n_se)
    s.set_scene(sc)
    for _ in range(5):
        s.solve()
    s.synchronize()
    print(json.dumps({"workload": args.workload, "K": p.K, "T": p.T, "n_obstacles": len(sc.obstacles),
                      "no_cull": bool(args.no_cull), "phase_us": s.get_phase_times()}))
    s.close()


def run_sweep(args):
    """BASELINE.json configs[4]: K x T x obstacle-count sweep and the 64-scene batch; one JSON line
    per point with the rollout kernel's device time and roofline fraction."""
    from paper_2508_05773_b200 import brmppi as B
    peak = N_SMS * ISSUE_PER_CLK_PER_SM * float(measured_peaks().get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6

    def point(name, scs, p, n_scenes):
        n_obs = len(scs[0].obstacles)
        times = {}
        for label, flags in (("cull", 0), ("no_cull", B.FLAG_NO_CULL)):
            s = B.Solver(p, n_scenes, max(n_obs, 1), flags)
            for i, sc in enumerate(scs):
                s.set_scene(sc, i)
            for _ in range(3):
                s.solve()
            s.synchronize()
            times[label] = s.time_kernels(20)
            s.close()
        ms_roll, ms_upd = times["cull"]
        work = n_scenes * p.K * p.T
        instr = algorithmic_instr_per_sample_step(n_obs, len(p.discs))
        print(json.dumps({"point": name, "K": p.K, "T": p.T, "n_obstacles": n_obs, "n_scenes": n_scenes,
                          "rollout_us": ms_roll * 1e3, "update_us": ms_upd * 1e3,
                          "sample_steps_per_s": work / (ms_roll * 1e-3),
                          "frac": work * instr / (ms_roll * 1e-3) / peak,
                          "rollout_us_no_cull": times["no_cull"][0] * 1e3,
                          "frac_no_cull": work * instr / (times["no_cull"][0] * 1e-3) / peak}), flush=True)

    for K in (1024, 16384, 131072, 1048576):
        for T in (50, 100):
            for n_obs in (8, 32, 64):
                sc = scenes.scene_static(0, n_obs, K=K, T=T)
                point("sweep", [sc], sc.params, 1)
    batch = scenes.scene_batch(64, 16384, 80)
    point("batch64", batch, batch[0].params.with_(seed=0), 64)


def run_project(args):
    """The closed-form projection (12) on its own (brmppi_project, NEXT row 1's kernel): the paper's per-solve
    count, 5000 rollouts x 120 steps = 600 000 problems with N_o = 8, device-resident, L2
    flushed between timed launches; one JSON line with the HBM roofline, the oracle beside it."""
    import time
    import numpy as np
    import torch
    from paper_2508_05773_b200 import brmppi as B
    from scenes.projection import projection_batch
    n, n_o = 600_000, 8
    d = n_o + 2
    P = projection_batch(7, n, n_o)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    A, b, zd = dev(P["A"]), dev(P["b"]), dev(P["z_des"])
    call = lambda: B.project(A, b, zd, P["w"], P["rho"], P["z_lo"], P["z_hi"])
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(max(args.warmup, 3)):
        call()
    ms = []
    for _ in range(args.steps):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        call()
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    t = float(np.mean(ms)) * 1e-3
    bytes_alg = n * 4 * (n_o * d + n_o + 2 * d)          # A, b, z_des in; z out
    mp = measured_peaks()
    peak = float(mp.get("hbm_gbs", 6500.0))
    # end to end through the C ABI with HOST buffers (page-locked) and a caller-owned device scratch: the call
    # copies A, b, z_des in and z out itself
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    hA, hb, hz = pin(P["A"]), pin(P["b"]), pin(P["z_des"])
    hout = torch.empty((n, d), dtype=torch.float32).pin_memory()
    scratch = torch.empty(B.lib().brmppi_project_scratch_bytes(n, n_o), dtype=torch.uint8, device="cuda")
    B.project(hA, hb, hz, P["w"], P["rho"], P["z_lo"], P["z_hi"], out=hout, scratch=scratch)
    reps = 5
    t0 = time.perf_counter()
    for _ in range(reps):
        B.project(hA, hb, hz, P["w"], P["rho"], P["z_lo"], P["z_hi"], out=hout, scratch=scratch)
    t_e2e = (time.perf_counter() - t0) / reps
    from oracle import projection as OP
    m = 20000
    t0 = time.perf_counter()
    for i in range(m):
        OP.project(P["A"][i], P["b"][i], P["z_des"][i], P["w"], P["rho"], P["z_lo"], P["z_hi"])
    t_cpu = time.perf_counter() - t0
    print(json.dumps({
        "metric": "brmppi_projections_per_s", "value": n / t, "unit": "projections/s", "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": t * 1e3, "higher_is_better": True,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "eq. (12), 5000 x 120 problems, N_o = 8 (PAPER.md:243)", "n": n, "n_o": n_o,
                   "l2": "flushed between timed launches (256 MiB write)"},
        "gpu_launches": args.steps,
        "e2e": {"value": n / t_e2e, "unit": "projections/s", "h2d_bytes_per_step": int(4 * (hA.numel() + hb.numel() + hz.numel())),
                "d2h_bytes_per_step": int(4 * hout.numel()), "what": "brmppi_project with page-locked host pointers and a "
                "caller-owned device scratch, host wall clock"},
        "roofline": {"bound": "hbm", "achieved": bytes_alg / t / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": bytes_alg / t / 1e9 / peak, "traffic": dram_traffic_from_profile("r1d_project_dram.csv")[0],
                     "traffic_source": dram_traffic_from_profile("r1d_project_dram.csv")[1], "kernel": "project_batch_bulk<8> (persistent; its last CTA takes the 64-problem tail)",
                     "algorithmic_bytes_per_problem": bytes_alg // n,
                     "peak_basis": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in mp else "fallback 6500 GB/s"},
        "cpu_baseline": {"value": m / t_cpu, "unit": "projections/s", "cores": 1, "kind": "oracle",
                         "sample": f"first {m} of the {n} problems, oracle/projection.py"}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg2se", "cfg3", "cfg2proj", "paperproj", "cfg2mpcc", "papermpcc"])
    ap.add_argument("--no-others", action="store_true", help="skip the secondary workloads of the `others` key")
    ap.add_argument("--phases", action="store_true", help="print the rollout kernel's in-kernel phase times")
    ap.add_argument("--sweep", action="store_true", help="run BASELINE.json configs[4] (sweep + 64-scene batch)")
    ap.add_argument("--project", action="store_true", help="time the closed-form projection (12) on its own")
    ap.add_argument("--sharded", action="store_true", help="K-sharded solve over the ranks (strong scaling) instead of replicas")
    ap.add_argument("--peaks", action="store_true", help="issue-rate micro-benchmarks (brmppi_measure_peaks): the dispatch-cost table")
    ap.add_argument("--no-cull", action="store_true", help="evaluate every (obstacle, disc, step): BRMPPI_FLAG_NO_CULL")
    args = ap.parse_args()
    if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) <= 1 and not (args.project or args.phases or args.sweep):
        spawn_ranks(args)          # reference arm included: rank 0 runs it, the others exit 0
    if args.peaks:
        from paper_2508_05773_b200 import brmppi as B
        pk = B.measure_peaks()
        pk["unit"] = "thread-instructions per clock per SM (128 = one warp instruction per clock per scheduler)"
        pk["cycles_per_warp_instruction_per_scheduler"] = {k: round(128.0 / v, 3) for k, v in pk.items()
                                                           if isinstance(v, float) and k not in ("sm_mhz", "sm_mhz_under_ffma") and v > 0}
        print(json.dumps(pk))
    elif args.project:
        run_project(args)
    elif args.phases:
        run_phases(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
