#!/usr/bin/env python
"""Benchmark of the batched fixed-lag SLAM backbone (BASELINE.json metric: env-steps/s + roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3|0|1|2|4:16384] [--impl reference]

One "step" = one pass of the whole hot path (push -> Gauss-Newton solve -> last-pose covariance and
log-det -> marginalisation) over the whole batch of environments = ONE fused kernel launch
(slam_step; landmark windows add a tiny second launch that orders the environments for the next step).  Default workload: BASELINE.json configs[3] (N=16384 envs, W=20 poses, L=24 landmarks,
2 GN iterations, 300 steps), the configuration the north_star's roofline target is quoted on.
Inputs are seeded synthetic trajectories (harness/synth.py), resident in HBM before
the timed region.  Rank 0 prints ONE JSON line.  Multi-GPU: environments are independent, so N ranks
run N replicas of the workload (different seeds) with no collective on the data path ("weak").
"""
from __future__ import annotations

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

from harness import replicas, synth, workmodel  # noqa: E402

SM_COUNT, LANES = 148, 128           # nominal unit counts (B200_PROFILING.md); the peak used is MEASURED, see fp32_peak()
L2_BYTES = 126 * 2 ** 20
METRIC = "fixed-lag SLAM env-steps/sec (solve+cov+marginalize)"
TRAFFIC_PROFILE = os.path.join(ROOT, "profiles", "r2_step_kernel_full.md")


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE steady-state slam_step_kernel launch, from the committed
    `ncu --set full` capture: the line `traffic_bytes_per_launch[<workload>] = <bytes>` of profiles/r2_step_kernel_full.md
    (None when the profile has no such line)."""
    import re
    try:
        for line in open(TRAFFIC_PROFILE):
            m = re.match(r"\s*traffic_bytes_per_launch\[(\w+)\]\s*=\s*([0-9.eE+]+)", line)
            if m and m.group(1) == workload:
                return float(m.group(2))
    except OSError:
        pass
    return None


def config_of(cfg, world: int, flush: bool, touched_mib: float) -> dict:
    """The `config` object of the JSON line; both arms (ours / --impl reference) print the same one."""
    return {"workload": cfg.name, "envs": cfg.N, "window": cfg.W, "landmarks": cfg.L, "gn_iters": cfg.iters,
            "p_loop_closure": cfg.p_lc, "parallelism": f"replicas x{world}, no collective",
            "l2": ("flushed between steps (untimed)" if flush else
                   f"not flushed: {touched_mib:.0f} MiB algorithmic working set per step > L2")}


def preroll_steps(cfg) -> int:
    """Untimed steps from reset before the timed region: the window is full (count == W at every timed solve,
    every timed step marginalises) and the prior has reached its steady-state support."""
    return cfg.W + 5


def touched_mib_of(cfg) -> float:
    """Rough algorithmic working set per batch step (record state + factor data + dense-ish prior support), only to
    decide whether the L2 has to be flushed between steps."""
    n = 3 * cfg.W + 2 * cfg.L
    per_env = 4.0 * (2 * n + 7 * cfg.W + 2 * cfg.W * cfg.L) + 4.0 * (0.35 * n) ** 2
    return per_env * cfg.N / 2 ** 20


def parse_config(s: str) -> synth.Config:
    if ":" in s:
        k, n = s.split(":")
        assert int(k) == 4, "only config 4 takes an N"
        return synth.config4(int(n))
    k = int(s)
    return synth.config4(16384) if k == 4 else synth.CONFIGS[k]


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        d["_source"] = "measured (MEASURED_PEAKS.json)"
        return d
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "_source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""

    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for nme, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(cfg, steps_total: int, seconds: float, threads: int) -> np.ndarray:
    """Environments (spread over the batch) the fp64 oracle can run for `steps_total` steps in about `seconds`."""
    n = 3 * cfg.W + 2 * cfg.L
    est = 2.2 * n ** 3 / 1.0e9                          # rough seconds per env-step per thread (measured)
    ne = int(max(threads, min(cfg.N, round(seconds * threads / (steps_total * est)))))
    return np.unique(np.linspace(0, cfg.N - 1, ne).astype(np.int32))


def cpu_oracle_leg(data, cfg, steps_total, seconds=15.0):
    """The fp64 oracle, as it stands, on the host cores, on a bounded sample of the same workload (all the steps
    the GPU ran: pre-roll + timed)."""
    import oracle
    threads = oracle.max_threads()
    envs = oracle_sample(cfg, steps_total, seconds, threads)
    t0 = time.perf_counter()
    res = oracle.run_batch(data, cfg.iters, envs=envs, want=("poses", "cov", "logdet"))
    dt = time.perf_counter() - t0
    return {"value": len(envs) * steps_total / dt, "unit": "env-steps/s", "cores": threads, "kind": "oracle",
            "sample": f"{len(envs)} of {cfg.N} envs x {steps_total} steps (pre-roll + timed), fp64 dense oracle, {dt:.1f} s"}, envs, res


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle timed on the host cores."""
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    import oracle
    cfg = parse_config(args.config)
    P = preroll_steps(cfg)
    K, Wm = args.steps or max(cfg.T - P, 1), args.warmup
    threads = oracle.max_threads()
    envs = oracle_sample(cfg, K, 60.0, threads)
    data = synth.generate(cfg, env_ids=envs, steps=K)
    if Wm > 0:
        warm = synth.generate(cfg, env_ids=envs[:threads], steps=min(Wm, K))
        oracle.run_batch(warm, cfg.iters, want=("logdet",))
    t0 = time.perf_counter()
    res = oracle.run_batch(data, cfg.iters, want=("logdet",))
    dt = time.perf_counter() - t0
    v = len(envs) * K / dt
    sample = f"{len(envs)} of {cfg.N} envs x {K} steps per run (from reset: the dense oracle's cost per step does not depend on the window count), fp64 dense oracle on {threads} threads"
    tm = touched_mib_of(cfg)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "env-steps/s", "n_gpus": args.gpus, "steps": K,
        "warmup": Wm, "ms_per_step": 1e3 * dt / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": config_of(cfg, world, tm * 2 ** 20 < 2 * L2_BYTES, tm),
        "cpu_baseline": {"value": v, "unit": "env-steps/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "env-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "singular_envs": int(res["bad"]),
    }))


def run_scan(args):
    """--config scan:N -- NEXT-3 (scan matcher + grid update) on N synthetic worlds; one step = match + update."""
    import torch
    from paper_2603_25834_b200 import binding
    from oracle import scanmatch as osm
    N = int(args.config.split(":")[1])
    K, Wm = args.steps or 20, max(args.warmup, 3)
    w = synth.generate_scan_world(N, seed=0, offset_cells=(1, -2, 2), range_sigma=0.01)
    par = binding.ScanParams(G=w["G"], res=w["res"], R=w["R"], r_min=0.1, r_max=10.0, hx=3, hy=3, ht=4, sxy=0.1, sth=0.01)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    grid0, pred, rng_ = dev(w["grid"]), dev(w["pose_pred"]), dev(w["ranges"])
    grid = grid0.clone()

    def step():
        meas, s1, s2 = binding.scan_match(par, grid, pred, rng_)
        binding.grid_update(par, grid, meas, rng_, s1, 0.4, 0.9, 5.0)
        return s1

    for _ in range(Wm):
        step()
    grid.copy_(grid0)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        e0.record()
        for _ in range(K):
            s1 = step()
        e1.record()
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    G, R = w["G"], w["R"]
    bytes_step = N * (3 * G * G * 4 + 2 * R * 4 + 40)       # grid: match read + clamp read/write; scans twice
    peaks = measured_peaks()
    t0 = time.perf_counter()
    ne = min(N, 8)
    for e in range(ne):
        m, o1, o2, _, _ = osm.scan_match(w["grid"][e].astype(np.float64), w["pose_pred"][:, e].astype(np.float64),
                                         w["ranges"][:, e].astype(np.float64), 0.1, 3, 3, 4, 0.1, 0.01)
        osm.grid_update(w["grid"][e].astype(np.float64), m, w["ranges"][:, e].astype(np.float64), o1, 0.1, 0.4, 0.9, 5.0)
    cpu_s = time.perf_counter() - t0
    achieved = bytes_step * K / (ms * 1e-3) / 1e9
    print(json.dumps({
        "metric": "scan-match + grid-update env-steps/sec (NEXT-3)", "value": N * K / (ms * 1e-3), "unit": "env-steps/s",
        "n_gpus": 1, "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 (fp64 cell decisions)", "data": "synthetic",
        "config": {"workload": f"scan_{N}", "envs": N, "grid": G, "rays": R, "candidates": 7 * 7 * 9,
                   "l2": f"{N * G * G * 4 / 2 ** 20:.0f} MiB of grids per step" },
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                     "frac": achieved / float(peaks["hbm_gbs"]), "traffic": None, "kernel": "scan_match_kernel + grid_update_kernel",
                     "alg_bytes_per_env_step": bytes_step / N},
        "clocks": clk.summary(), "gpu_launches": 3 * K,
        "cpu_baseline": {"value": ne / cpu_s, "unit": "env-steps/s", "cores": 1, "kind": "oracle",
                         "sample": f"{ne} envs, numpy/python fp64 oracle, {cpu_s:.1f} s"},
        "mean_score": float(s1.mean().item()),
    }))


def fp32_peak(device, seconds=0.25) -> dict:
    """FP32 FMA peak MEASURED on this GPU with the library's register-resident microbenchmark (slam_fma_probe):
    best of several launches, CUDA events on the launching stream, SM clock sampled while it runs."""
    import torch
    from paper_2603_25834_b200 import binding
    iters = 4096
    binding.fma_probe(64, device)                       # module load + warm-up
    torch.cuda.synchronize(device)
    best, flops = 0.0, 0.0
    with ClockSampler(device.index or 0) as clk:
        t_end = time.perf_counter() + seconds
        while True:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            flops = binding.fma_probe(iters, device)
            e1.record()
            torch.cuda.synchronize(device)
            best = max(best, flops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
            if time.perf_counter() > t_end:
                break
    return {"tflops": best, "sm_mhz": clk.summary()["sm_mhz"], "flops_per_launch": flops}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0,
                    help="batch steps to time in steady state (default: the config's step count minus the pre-roll)")
    ap.add_argument("--warmup", type=int, default=3, help="untimed warm-up steps (the pre-roll to a full window covers them)")
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the timed region (median and best are reported)")
    ap.add_argument("--config", default="3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--flush-l2", choices=["auto", "on", "off"], default="auto")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-all-steps", action="store_true", help="skip the extra from-reset run (window-fill phase included)")
    ap.add_argument("--work-sample", type=int, default=256, help="environments the algorithmic work model replays")
    args = ap.parse_args()
    if args.config.startswith("scan:"):
        return run_scan(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2603_25834_b200.binding import FixedLagSlam

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    device = torch.device(f"cuda:{local}")

    base = parse_config(args.config)
    cfg = synth.Config(base.name, base.N, base.W, base.L, base.iters, base.T, base.p_lc, seed=replicas.rank_seed(base.seed, rank))
    # Timed region = K consecutive STEADY-STATE steps: P untimed steps from reset first (window full, prior at its
    # steady support; P >= the requested warm-up), so every timed step is push + solve + covariance + marginalise
    # on a full window -- what the metric names.  The from-reset run (window-fill phase included) is reported
    # separately as `all_steps`.
    P = max(preroll_steps(cfg), args.warmup)
    K = args.steps or max(cfg.T - P, 1)
    Wm = max(args.warmup, 0)
    T_tot = P + K
    R = max(args.reps, 1)
    N, W, L, nw = cfg.N, cfg.W, cfg.L, (cfg.L + 31) // 32
    data = synth.generate(cfg, steps=T_tot)
    dev = {k: torch.from_numpy(np.ascontiguousarray(data[k] if k != "rb_mask" else data[k].view(np.int32))).to(device)
           for k in ("odom", "lc_back", "lc_meas", "rb_mask", "rb_meas")}
    slam = FixedLagSlam(N, W, L, device=device)
    cov = torch.zeros(T_tot, 9, N, device=device)
    logdet = torch.zeros(T_tot, N, device=device)
    last_pose = torch.zeros(T_tot, 3, N, device=device)

    def args_of(t):
        return (dev["odom"][t - 1], dev["lc_back"][t - 1], dev["lc_meas"][t - 1],
                dev["rb_mask"][t] if L else None, dev["rb_meas"][t] if L else None)

    def step(t):
        slam.step(*args_of(t), iters=cfg.iters, cov=cov[t - 1], logdet=logdet[t - 1], last_pose=last_pose[t - 1])

    def start(upto=0):
        """reset, then steps 1..upto untimed"""
        slam.reset()
        if L:
            slam.observe_first(dev["rb_mask"][0], dev["rb_meas"][0])
        for t in range(1, upto + 1):
            step(t)

    # algorithmic work of the timed steps (sampled environments; structure only, host logic)
    sample = np.unique(np.linspace(0, N - 1, min(N, max(args.work_sample, 1))).astype(np.int64))
    work = workmodel.step_work_parallel(data, cfg.iters, sample, steps=T_tot, procs=min(16, os.cpu_count() or 1))
    flops_total = float(work["flops"][P:].sum()) * N
    bytes_total = float(work["bytes"][P:].sum()) * N
    tm = touched_mib_of(cfg)
    flush = args.flush_l2 == "on" or (args.flush_l2 == "auto" and tm * 2 ** 20 < 2 * L2_BYTES)
    scratch = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=device) if flush else None

    def barrier():
        replicas.barrier(world)

    def timed(t_first, t_last):
        """device milliseconds of steps t_first..t_last (CUDA events on the launching stream)"""
        if flush:   # per-step events, L2 flushed (untimed) between steps
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(t_first, t_last + 1)]
            for i, t in enumerate(range(t_first, t_last + 1)):
                scratch.fill_(t & 0xFF)
                evs[i][0].record()
                step(t)
                evs[i][1].record()
            torch.cuda.synchronize()
            return sum(a.elapsed_time(b) for a, b in evs)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(t_first, t_last + 1):
            step(t)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    peak = fp32_peak(device) if rank == 0 else None

    # ---- steady state: R repetitions of [reset, P untimed steps, K timed steps]
    reps_ms, ktime, launches = [], None, 0
    barrier()
    with ClockSampler(local) as clk:
        for r in range(R):
            start(P)
            torch.cuda.synchronize()
            if r == R - 1:
                slam.kernel_timing(K)               # per-kernel events of the last repetition (library side)
            l0 = slam.launch_count
            barrier()
            reps_ms.append(timed(P + 1, T_tot))
            launches = slam.launch_count - l0
            barrier()
    ktime = slam.kernel_timing_read()
    slam.kernel_timing(0)
    stats = slam.get_stats()
    status_bad = int((slam.get_status() != 0).sum().item())
    finite = bool(torch.isfinite(logdet).all().item() and torch.isfinite(cov).all().item())
    ms_med, ms_best = statistics.median(reps_ms), min(reps_ms)

    # ---- all steps from reset (window-fill phase included), the other number SURVEY.md 8(d) asks for
    all_ms = None
    T_all = min(cfg.T, T_tot)
    if not args.no_all_steps:
        runs = []
        for r in range(2):
            start(0)
            torch.cuda.synchronize()
            barrier()
            runs.append(timed(1, T_all))
        all_ms = min(runs)       # (the same trajectory: cov / logdet / last_pose hold the same values as before)

    # ---- end to end through the host-buffer entry point (pinned inputs, outputs copied back every step)
    e2e = None
    if not args.no_e2e:
        # slices [P:]: index i = timed step P + 1 + i for odom / lc_*, index i + 1 for the range-bearing arrays
        pin = {k: torch.from_numpy(np.ascontiguousarray(data[k][P:] if k != "rb_mask" else data[k][P:].view(np.int32))).pin_memory()
               for k in ("odom", "lc_back", "lc_meas", "rb_mask", "rb_meas")}
        hcov, hld, hpose = torch.zeros(9, N).pin_memory(), torch.zeros(N).pin_memory(), torch.zeros(3, N).pin_memory()
        start(P)
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for i in range(K):
            slam.step_host(pin["odom"][i], pin["lc_back"][i], pin["lc_meas"][i],
                           pin["rb_mask"][i + 1] if L else None, pin["rb_meas"][i + 1] if L else None,
                           iters=cfg.iters, cov=hcov, logdet=hld, last_pose=hpose)
            slam.stream.synchronize()          # the caller reads this step's covariance / log-det / pose
        e2e_s = time.perf_counter() - t0
        barrier()
        e2e = {"seconds": e2e_s, "h2d": N * 4 * (3 + 1 + 3 + nw + 2 * L), "d2h": N * 4 * 13}

    # max over ranks (device-timed)
    ms_max, ms_best_max, e2e_s_max, all_ms_max = replicas.max_over_ranks(
        [ms_med, ms_best, e2e["seconds"] if e2e else 0.0, all_ms or 0.0], world, device)
    value = replicas.whole_job_rate(N * K, world, ms_max * 1e-3)

    if rank == 0:
        peaks = measured_peaks()
        clocks = clk.summary()
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        p_nominal = SM_COUNT * LANES * 2 * sm_max * 1e6 / 1e12               # TFLOP/s, plain FP32 FMA issue peak
        p_fp32 = peak["tflops"]
        bw = float(peaks["hbm_gbs"])
        t_meas = ms_med * 1e-3
        t_alu, t_hbm = flops_total / (p_fp32 * 1e12), bytes_total / (bw * 1e9)
        bound = "alu" if t_alu >= t_hbm else "hbm"
        ksteps = max(ktime["steps"], 1)
        k_step, k_ref, k_ord = ktime["step_kernel_ms"] / ksteps, ktime["ref64_kernel_ms"] / ksteps, ktime["order_kernel_ms"] / ksteps
        roof = {"bound": bound, "unit": "TFLOP/s" if bound == "alu" else "GB/s",
                "achieved": (flops_total / t_meas / 1e12) if bound == "alu" else (bytes_total / t_meas / 1e9),
                "peak": p_fp32 if bound == "alu" else bw,
                "frac": max(t_alu, t_hbm) / t_meas, "traffic": ncu_traffic(cfg.name),
                "kernel": "slam_step_kernel", "kernel_ms_avg": k_step,
                "kernels_ms_avg": {"slam_step_kernel": k_step, "slam_ref64_kernel": k_ref, "slam_order_kernel": k_ord},
                "step_kernel_share": k_step / max(k_step + k_ref + k_ord, 1e-12),
                "denominator": "whole step (all its launches), median repetition; the algorithmic work of a step is "
                               "done by slam_step_kernel, except the ill-conditioned environments slam_ref64_kernel redoes",
                "alg_flops_per_env_step": flops_total / (N * K), "alg_bytes_per_env_step": bytes_total / (N * K),
                "alu_frac": t_alu / t_meas, "hbm_frac": t_hbm / t_meas,
                "fp32_tflops_measured": p_fp32, "fp32_probe_sm_mhz": peak["sm_mhz"], "fp32_tflops_nominal": p_nominal,
                "frac_of_nominal": flops_total / (p_nominal * 1e12) / t_meas,
                "peak_source": f"FP32: measured, slam_fma_probe ({SM_COUNT * 8} CTAs x 256 threads x 16 FMA chains), best launch; "
                               f"nominal {SM_COUNT} SMs x {LANES} lanes x 2 x {sm_max:.0f} MHz beside it; "
                               f"HBM {bw:.0f} GB/s {peaks['_source']}",
                "work_sample_envs": int(len(sample)),
                "envelope_words_avg": float(work["env_words"][P:].mean()), "prior_support_avg": float(work["support"][P:].mean()),
                "fp64_env_calls_frac": stats["fp64_calls"] / max(stats["solved"] + stats["fp64_calls"], 1)}
        # the dominant kernel ALONE: the algorithmic flops of the environments it solved over its own launch time
        # (`frac` above charges the whole step, fp64 and ordering launches included, to the same flops)
        roof["frac_step_kernel_alone"] = (flops_total / K * (1.0 - roof["fp64_env_calls_frac"])) / \
            max(k_step * 1e-3, 1e-12) / (p_fp32 * 1e12)
        out = {
            "metric": METRIC, "value": value, "unit": "env-steps/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": config_of(cfg, world, flush, tm),
            "timing": {"phase": "steady state", "preroll_steps": P, "full_window_steps": K, "reps": R,
                       "median_ms_per_step": ms_max / K, "best_ms_per_step": ms_best_max / K,
                       "reps_ms_per_step": [x / K for x in reps_ms]},
            "roofline": roof, "clocks": clocks, "gpu_launches": launches,
            "status_flagged_envs": status_bad, "outputs_finite": finite,
            "kernel_info": dict(slam.kernel_info(), pool_waits=stats["waited"]),
        }
        if all_ms is not None:
            out["all_steps"] = {"phase": "from reset, window-fill phase included", "steps": T_all, "ms_per_step": all_ms_max / T_all,
                                "value": replicas.whole_job_rate(N * T_all, world, all_ms_max * 1e-3), "best_of": 2}
        if e2e:
            out["e2e"] = {"value": replicas.whole_job_rate(N * K, world, e2e_s_max), "unit": "env-steps/s",
                          "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"]}
        if not args.no_cpu_baseline and world == 1:
            from tests.gpu_driver import parity_errors
            cb, envs, res = cpu_oracle_leg(data, cfg, T_tot)
            out["cpu_baseline"] = cb
            # parity of the run itself on the sampled environments, all steps (oracle values; R23 tolerances)
            ix = torch.from_numpy(envs.astype(np.int64)).to(device)
            gpu = {"cov": cov[:, :, ix].cpu().numpy().reshape(T_tot, 3, 3, len(envs)).transpose(0, 3, 1, 2).astype(np.float64),
                   "logdet": logdet[:, ix].cpu().numpy().astype(np.float64),
                   "last_pose": last_pose[:, :, ix].cpu().numpy().transpose(0, 2, 1).astype(np.float64)}
            err = parity_errors(gpu, res)
            worst = np.max([err[k] for k in err], axis=0)
            out["parity_sampled"] = {"envs": int(len(envs)), "env_steps": int(worst.size),
                                     "tolerances": "pose rel 1e-4, cov 1e-3 sqrt(S_ii S_jj), ln det abs 1e-3 (DESIGN.md R23)",
                                     "frac_within_tol": float((worst <= 1.0).mean()),
                                     "worst_over_tol": {k: float(err[k].max()) for k in err},
                                     "ok": bool((worst <= 1.0).mean() >= 0.999)}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
