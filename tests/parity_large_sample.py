"""Parity of config 3 on a LARGE sample, beyond what the test suite can afford.

    python tests/parity_large_sample.py [stride=4] [hi:lo:min_vis ...]

Runs the fp64 oracle on every `stride`-th environment of BASELINE config 3 (stride 4: 4096 environments x 300 steps,
about three minutes on 16 host threads), then the full batch on cuda:0 through the C ABI -- first with every environment
on the fp64 kernel (the device reference), then once per setting `hi:lo:min_vis` of the fp32 -> fp64 switch
(default: the library's 300:150:3 and the pivot ratio alone, 300:150:0) -- and prints, per run, the share of the
environment-calls that went through the fp64 kernel, the worst error in units of the tolerances of R23, how many
env-steps are beyond them, and for each of those the device reference's error at the same (step, environment).
A developer tool: it asserts nothing; the tests that pin its findings are in tests/test_gpu_parity.py."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import oracle
    from harness import synth
    from paper_2603_25834_b200.binding import FixedLagSlam
    from tests.gpu_driver import parity_errors, run_gpu

    stride = int(sys.argv[1]) if len(sys.argv) > 1 else 4
    settings = [tuple(float(x) for x in a.split(":")) for a in sys.argv[2:]] or [(300, 150, 3), (300, 150, 0)]   # hi:lo:min_vis[:box_vis]
    cfg = synth.CONFIGS[3]
    data = synth.generate(cfg)
    envs = np.arange(0, cfg.N, stride, dtype=np.int32)
    t0 = time.time()
    ref = oracle.run_batch(data, cfg.iters, envs=envs)
    print(f"oracle: {len(envs)} environments x {cfg.T} steps in {time.time() - t0:.0f} s", flush=True)

    def sub(g):
        return {k: (v[:, envs] if v.ndim >= 2 and v.shape[1] == cfg.N else v) for k, v in g.items()}

    def report(name, slam, g):
        err = parity_errors(g, ref)
        st = slam.get_stats()
        line = [f"{name}: fp64 calls {st['fp64_calls'] / (cfg.N * cfg.T):.4f}"]
        for k, v in err.items():
            line.append(f"{k} max {v.max():.3f}, {int((v > 1).sum())} of {v.size} beyond tolerance ({int((v > 0.5).sum())} beyond half of it)")
        print(" | ".join(line), flush=True)
        return err

    slam = FixedLagSlam(cfg.N, cfg.W, cfg.L, device="cuda:0")
    slam.set_precision(2)
    g64 = sub(run_gpu(slam, data, cfg.iters, fused=True, want_poses=False))
    e64 = report("device reference (every environment in fp64)", slam, g64)
    del slam
    for st_ in settings:
        hi, lo, mv = st_[:3]
        os.environ["SLAM_RATIO_HI"], os.environ["SLAM_RATIO_LO"], os.environ["SLAM_MIN_VIS"] = str(hi), str(lo), str(int(mv))
        if len(st_) > 3:
            os.environ["SLAM_BOX_VIS"] = str(int(st_[3]))
        slam = FixedLagSlam(cfg.N, cfg.W, cfg.L, device="cuda:0")
        g = sub(run_gpu(slam, data, cfg.iters, fused=True, want_poses=False))
        err = report(f"ratio_hi {hi:g} ratio_lo {lo:g} min_vis {int(mv)}" + (f" box_vis {int(st_[3])}" if len(st_) > 3 else ""), slam, g)
        bad = np.argwhere((err["logdet"] > 1) | (err["cov"] > 1) | (err["last_pose"] > 1))
        for t, i in bad[:60]:
            print(f"    step {int(t) + 1} env {int(envs[i])}: ln det {err['logdet'][t, i]:.2f} cov {err['cov'][t, i]:.2f} "
                  f"pose {err['last_pose'][t, i]:.2f} | device reference: ln det {e64['logdet'][t, i]:.3f} cov {e64['cov'][t, i]:.3f}")
        del slam


if __name__ == "__main__":
    main()
