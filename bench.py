#!/usr/bin/env python
"""Benchmark of the batched fixed-lag SLAM backbone (BASELINE.json metric: env-steps/s + roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3|0|1|2|4:16384] [--impl reference]

One "step" = one pass of the whole hot path (push -> Gauss-Newton solve -> last-pose covariance and
log-det -> marginalisation) over the whole batch of environments = ONE fused kernel launch
(slam_step; landmark windows add a tiny second launch that orders the environments for the next step).  Default workload: BASELINE.json configs[3] (N=16384 envs, W=20 poses, L=24 landmarks,
2 GN iterations, 300 steps), the configuration the north_star's roofline target is quoted on.
Inputs are seeded synthetic trajectories (paper_2603_25834_b200/synth.py), resident in HBM before
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

from paper_2603_25834_b200 import replicas, synth, workmodel  # noqa: E402

SM_COUNT, LANES = 148, 128
# dram__bytes_read.sum + dram__bytes_write.sum of one slam_step_kernel launch from the committed
# `ncu --set full` capture (profiles/r1e_step_kernel_full.md), keyed by workload
NCU_TRAFFIC_BYTES = {"cfg3_landmarks_16384": 169.1e6}
L2_BYTES = 126 * 2 ** 20
METRIC = "fixed-lag SLAM env-steps/sec (solve+cov+marginalize)"


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


def cpu_oracle_leg(data, cfg, K, seconds=15.0):
    """The fp64 oracle, as it stands, on the host cores, on a bounded sample of the same workload."""
    import oracle
    threads = oracle.max_threads()
    n = 3 * cfg.W + 2 * cfg.L
    est = 2.2 * n ** 3 / 1.0e9                          # rough seconds per env-step per thread (measured)
    ne = int(max(threads, min(cfg.N, round(seconds * threads / (K * est)))))
    envs = np.unique(np.linspace(0, cfg.N - 1, ne).astype(np.int32))
    t0 = time.perf_counter()
    res = oracle.run_batch(data, cfg.iters, envs=envs, want=("cov", "logdet"))
    dt = time.perf_counter() - t0
    probe = oracle.run_batch(data, cfg.iters, envs=envs, want=("logdet",), f32_storage=True)   # untimed: conditioning probe
    res["probe_logdet"] = probe["logdet"]
    return {"value": len(envs) * K / dt, "unit": "env-steps/s", "cores": threads, "kind": "oracle",
            "sample": f"{len(envs)} of {cfg.N} envs x all {K} steps, fp64 dense oracle, {dt:.1f} s"}, envs, res


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle timed on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = parse_config(args.config)
    K, Wm = args.steps or cfg.T, args.warmup
    threads = oracle.max_threads()
    n = 3 * cfg.W + 2 * cfg.L
    est = 2.2 * n ** 3 / 1.0e9
    ne = int(max(threads, min(cfg.N, round(60.0 * threads / (K * est)))))
    envs = np.unique(np.linspace(0, cfg.N - 1, ne).astype(np.int32))
    data = synth.generate(cfg, env_ids=envs, steps=K)
    if Wm > 0:
        warm = synth.generate(cfg, env_ids=envs[:threads], steps=min(Wm, K))
        oracle.run_batch(warm, cfg.iters, want=("logdet",))
    t0 = time.perf_counter()
    res = oracle.run_batch(data, cfg.iters, want=("logdet",))
    dt = time.perf_counter() - t0
    v = len(envs) * K / dt
    sample = f"{len(envs)} of {cfg.N} envs x {K} steps per run, fp64 dense oracle on {threads} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "env-steps/s", "n_gpus": args.gpus, "steps": K,
        "warmup": Wm, "ms_per_step": 1e3 * dt / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "envs": cfg.N, "window": cfg.W, "landmarks": cfg.L, "gn_iters": cfg.iters,
                   "sampled_envs": len(envs)},
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="batch steps to time (default: the config's step count)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--flush-l2", choices=["auto", "on", "off"], default="auto")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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
    K = args.steps or cfg.T
    Wm = max(args.warmup, 0)
    N, W, L, nw = cfg.N, cfg.W, cfg.L, (cfg.L + 31) // 32
    data = synth.generate(cfg, steps=K)
    dev = {k: torch.from_numpy(np.ascontiguousarray(data[k] if k != "rb_mask" else data[k].view(np.int32))).to(device)
           for k in ("odom", "lc_back", "lc_meas", "rb_mask", "rb_meas")}
    slam = FixedLagSlam(N, W, L, device=device)
    cov = torch.zeros(K, 9, N, device=device)
    logdet = torch.zeros(K, N, device=device)

    def args_of(t):
        return (dev["odom"][t - 1], dev["lc_back"][t - 1], dev["lc_meas"][t - 1],
                dev["rb_mask"][t] if L else None, dev["rb_meas"][t] if L else None)

    def start():
        slam.reset()
        if L:
            slam.observe_first(dev["rb_mask"][0], dev["rb_meas"][0])

    # algorithmic work of the timed steps (sampled environments; structure only)
    sample = np.unique(np.linspace(0, N - 1, min(N, 24)).astype(np.int64))
    work = workmodel.step_work(data, cfg.iters, sample, steps=K)
    flops_total = float(work["flops"].sum()) * N
    bytes_total = float(work["bytes"].sum()) * N
    touched_per_step = float(work["bytes"].mean()) * N
    flush = args.flush_l2 == "on" or (args.flush_l2 == "auto" and touched_per_step < 2 * L2_BYTES)
    scratch = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=device) if flush else None

    # warm-up (untimed), then restart the trajectory
    start()
    for t in range(1, min(Wm, K) + 1):
        slam.step(*args_of(t), iters=cfg.iters, cov=cov[t - 1], logdet=logdet[t - 1])
    torch.cuda.synchronize()
    start()
    launches0 = slam.launch_count

    def barrier():
        replicas.barrier(world)

    barrier()
    with ClockSampler(local) as clk:
        if flush:   # per-step events, L2 flushed (untimed) between steps
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
            for t in range(1, K + 1):
                scratch.fill_(t & 0xFF)
                evs[t - 1][0].record()
                slam.step(*args_of(t), iters=cfg.iters, cov=cov[t - 1], logdet=logdet[t - 1])
                evs[t - 1][1].record()
            torch.cuda.synchronize()
            ms = sum(a.elapsed_time(b) for a, b in evs)
        else:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for t in range(1, K + 1):
                slam.step(*args_of(t), iters=cfg.iters, cov=cov[t - 1], logdet=logdet[t - 1])
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
    barrier()
    launches = slam.launch_count - launches0
    status_bad = int((slam.get_status() != 0).sum().item())
    finite = bool(torch.isfinite(logdet).all().item())

    # end-to-end through the host-buffer entry point (pinned inputs, outputs copied back every step)
    e2e = None
    if not args.no_e2e:
        pin = {k: torch.from_numpy(np.ascontiguousarray(data[k] if k != "rb_mask" else data[k].view(np.int32))).pin_memory()
               for k in ("odom", "lc_back", "lc_meas", "rb_mask", "rb_meas")}
        hcov, hld = torch.zeros(9, N).pin_memory(), torch.zeros(N).pin_memory()
        start()
        barrier()
        t0 = time.perf_counter()
        for t in range(1, K + 1):
            slam.step_host(pin["odom"][t - 1], pin["lc_back"][t - 1], pin["lc_meas"][t - 1],
                           pin["rb_mask"][t] if L else None, pin["rb_meas"][t] if L else None,
                           iters=cfg.iters, cov=hcov, logdet=hld)
            slam.stream.synchronize()          # the caller reads this step's covariance / log-det
        e2e_s = time.perf_counter() - t0
        barrier()
        e2e = {"seconds": e2e_s, "h2d": N * 4 * (3 + 1 + 3 + nw + 2 * L), "d2h": N * 4 * 10}

    # max over ranks (device-timed)
    ms_max, e2e_s_max = replicas.max_over_ranks([ms, e2e["seconds"] if e2e else 0.0], world, device)
    value = replicas.whole_job_rate(N * K, world, ms_max * 1e-3)

    if rank == 0:
        peaks = measured_peaks()
        clocks = clk.summary()
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        p_fp32 = SM_COUNT * LANES * 2 * sm_max * 1e6 / 1e12                 # TFLOP/s, plain FP32 FMA issue peak
        bw = float(peaks["hbm_gbs"])
        t_meas = ms * 1e-3
        t_alu, t_hbm = flops_total / (p_fp32 * 1e12), bytes_total / (bw * 1e9)
        bound = "alu" if t_alu >= t_hbm else "hbm"
        roof = {"bound": bound, "unit": "TFLOP/s" if bound == "alu" else "GB/s",
                "achieved": (flops_total / t_meas / 1e12) if bound == "alu" else (bytes_total / t_meas / 1e9),
                "peak": p_fp32 if bound == "alu" else bw,
                "frac": max(t_alu, t_hbm) / t_meas, "traffic": NCU_TRAFFIC_BYTES.get(cfg.name),
                "kernel": "slam_step_kernel", "kernel_ms_avg": ms / K,
                "alg_flops_per_env_step": flops_total / (N * K), "alg_bytes_per_env_step": bytes_total / (N * K),
                "alu_frac": t_alu / t_meas, "hbm_frac": t_hbm / t_meas,
                "peak_source": f"FP32: {SM_COUNT} SMs x {LANES} lanes x 2 x {sm_max:.0f} MHz (derived, DESIGN.md); "
                               f"HBM {bw:.0f} GB/s {peaks['_source']}",
                "envelope_words_avg": float(work["env_words"].mean()), "prior_support_avg": float(work["support"].mean())}
        out = {
            "metric": METRIC, "value": value, "unit": "env-steps/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "envs": N, "window": W, "landmarks": L, "gn_iters": cfg.iters,
                       "p_loop_closure": cfg.p_lc, "parallelism": f"replicas x{world}, no collective",
                       "l2": ("flushed between steps (untimed)" if flush else
                              f"not flushed: {touched_per_step / 2 ** 20:.0f} MiB algorithmic working set per step > L2")},
            "roofline": roof, "clocks": clocks, "gpu_launches": launches,
            "status_flagged_envs": status_bad, "outputs_finite": finite,
            "kernel_info": dict(slam.kernel_info(), pool_waits=slam.get_stats()["waited"]),
        }
        if e2e:
            out["e2e"] = {"value": replicas.whole_job_rate(N * K, world, e2e_s_max), "unit": "env-steps/s",
                          "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"]}
        if not args.no_cpu_baseline and world == 1:
            cb, envs, res = cpu_oracle_leg(data, cfg, K)
            out["cpu_baseline"] = cb
            # parity of the timed run itself on the sampled environments (oracle values; R23 tolerances)
            g_ld = logdet[:, torch.from_numpy(envs.astype(np.int64)).to(device)].cpu().numpy().astype(np.float64)
            e_ld = np.abs(g_ld - res["logdet"])
            p_ld = np.abs(res["probe_logdet"] - res["logdet"])          # error of fp32 STORAGE alone (oracle probe)
            forked = np.maximum.accumulate(p_ld > 1e-3 / 12.0, axis=0)  # per env: from its first ill-conditioned step on
            out["parity_sampled"] = {"envs": int(len(envs)), "env_steps": int(e_ld.size), "tol_abs_logdet": 1e-3,
                                     "frac_within_tol": float((e_ld <= 1e-3).mean()),
                                     "strict_coverage": float((~forked).mean()),
                                     "max_err_well_conditioned": float(e_ld[~forked].max()) if (~forked).any() else None,
                                     "max_err_forked": float(e_ld[forked].max()) if forked.any() else 0.0,
                                     "probe_max_err": float(p_ld.max())}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
