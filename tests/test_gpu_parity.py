"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on identical seeded inputs.

Tolerances are BASELINE.json north_star's, in the reading R23 of DESIGN.md (written in
tests/gpu_driver.parity_errors): poses rel 1e-4, covariance 1e-3 of sqrt(S_ii S_jj), ln det abs 1e-3.
"""
import numpy as np
import pytest
import torch

import oracle
from harness import synth
from tests.gpu_driver import parity_errors, run_gpu, to_dev
from tests.helpers import determined, drive

pytestmark = pytest.mark.gpu


def _slam(N, W, L, precision=None):
    from paper_2603_25834_b200.binding import FixedLagSlam
    slam = FixedLagSlam(N, W, L)
    if precision is not None:
        slam.set_precision(precision)
    return slam


def _fused_equals_separate(cfg, data, ref=None):
    """slam_step against the composition of the separate calls.  Bit for bit while an environment stays in one
    precision mode (0: the fp32 kernel, 2: the fp64 kernel); with the conditioning watch on (mode 1) the fused call
    sees all its factorisations at once and the separate calls one at a time, so an environment near the threshold
    may change hands at a different call: both then hold the stated tolerances, not the same bits."""
    for mode in (0, 2):
        a = run_gpu(_slam(cfg.N, cfg.W, cfg.L, mode), data, cfg.iters, fused=False, want_poses=False)
        b = run_gpu(_slam(cfg.N, cfg.W, cfg.L, mode), data, cfg.iters, fused=True, want_poses=False)
        assert np.array_equal(a["cov"], b["cov"]) and np.array_equal(a["logdet"], b["logdet"]), mode
        c = run_gpu(_slam(cfg.N, cfg.W, cfg.L, mode), data, cfg.iters, fused=True, want_poses=False)   # and launch to launch
        assert np.array_equal(b["cov"], c["cov"]) and np.array_equal(b["last_pose"], c["last_pose"]), mode
    if ref is not None:
        b = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
        _check(b, ref, what=("cov", "logdet"))


def _check(gpu, ref, what=("poses", "last_pose", "cov", "logdet"), det=None, min_determined=0.999):
    """Every (step, env) must be within the stated tolerances R23 (error <= 1.0 in tolerance units).  `det` (config 3
    only): the env-steps the ORACLE itself determines (tests/helpers.determined: its outputs do not move when one
    input changes by one float32 ulp); at least 99.9 % must be, the others are not compared.

    Windows whose information matrix fp32 cannot carry (config 3 after the robot left the landmark box and
    re-observes a landmark) are recognised by the library's own conditioning watch and solved by its fp64 kernel
    (slam_set_precision): the test does not know about them."""
    err = parity_errors(gpu, ref)
    keys = [k for k in what if k in err]
    assert keys
    G = np.max([err[k] for k in keys], axis=0)
    assert np.isfinite(G).all()
    if det is not None:
        assert det.mean() >= min_determined, f"only {det.mean():.5f} of the env-steps are determined by the oracle"
        G = np.where(det, G, 0.0)
    worst = float(G.max())
    assert worst <= 1.0, f"{worst:.3g} x tolerance at (step, env) {np.unravel_index(G.argmax(), G.shape)}: " + \
        ", ".join(f"{k} {float(err[k].max()):.3g}" for k in keys)
    return err


def _sub(gpu, envs):
    return {k: (v[:, envs] if k != "status" else v[envs]) for k, v in gpu.items()}


def _window_after_step(slam, ref, t, envs=None, det=None):
    """slam_get_poses after the fused step t (1-based) against the oracle's window of that step: marginalisation
    only re-expresses the window in the next anchor's frame, so the global poses of the slots that stay are
    unchanged (oracle slots 1.. of step t = library slots 0.. after the step, once the window is full)."""
    W = slam.W
    P = slam.get_poses().cpu().numpy().transpose(2, 1, 0).astype(np.float64)     # [N, W, 3]
    if envs is not None:
        P = P[envs]
    R = ref["poses"][t - 1]                                                        # [ne, W, 3] after the solve of step t
    c = min(t + 1, W)
    if c == W:
        got, exp = P[:, : W - 1], R[:, 1:W]
    else:
        got, exp = P[:, :c], R[:, :c]
    d = got - exp
    d[..., 2] = np.arctan2(np.sin(d[..., 2]), np.cos(d[..., 2]))
    scale = np.maximum(1.0, np.abs(R).max(axis=(1, 2)))
    e = np.abs(d).max(axis=(1, 2)) / (1e-4 * scale)
    if det is not None:
        e = np.where(det[t - 1], e, 0.0)
    worst = float(e.max())
    assert worst <= 1.0, f"window poses after step {t}: {worst:.3g} x tolerance (env index {int(e.argmax())})"


def test_config0_all_envs_all_steps():
    cfg = synth.CONFIGS[0]
    data = synth.generate(cfg)
    ref = oracle.run_batch(data, cfg.iters)
    gpu = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref)
    fused = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    _check(fused, ref, what=("last_pose", "cov", "logdet"))


@pytest.mark.parametrize("W,L,p_lc,N,T,iters", [
    (6, 0, 0.4, 37, 60, 3),      # loops, ragged batch (not a multiple of the warps per CTA)
    (5, 7, 0.3, 33, 50, 2),      # landmarks + loops
    (2, 3, 0.0, 5, 20, 2),       # minimum window
    (8, 33, 0.2, 9, 40, 2),      # two visibility mask words
    (12, 1, 0.5, 1, 40, 3),      # single env, single landmark
    (64, 0, 0.2, 3, 100, 2),     # maximum window
    (4, 64, 0.0, 3, 30, 2),      # maximum landmarks
    (64, 64, 0.1, 2, 68, 2),     # maximum window AND landmarks: one team per CTA, the pool holds exactly one window
])
def test_small_cases_every_env(W, L, p_lc, N, T, iters):
    cfg = synth.Config("t", N=N, W=W, L=L, iters=iters, T=T, p_lc=p_lc, seed=3)
    data = synth.generate(cfg)
    ref = oracle.run_batch(data, iters)
    assert ref["bad"] == 0
    gpu = run_gpu(_slam(N, W, L), data, iters, fused=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref)


@pytest.mark.parametrize("W,L,p_lc", [(7, 0, 0.4), (6, 9, 0.3)])
def test_fused_step_is_bitwise_the_composition(W, L, p_lc):
    cfg = synth.Config("f", N=70, W=W, L=L, iters=2, T=40, p_lc=p_lc, seed=8)
    data = synth.generate(cfg)
    _fused_equals_separate(cfg, data, oracle.run_batch(data, cfg.iters))


def test_noise_free_recovers_ground_truth():
    cfg = synth.Config("nf", N=64, W=10, L=12, iters=2, T=60, p_lc=0.3, seed=5)
    data = synth.generate(cfg, noise_scale=0.0)
    gpu = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=False)
    for t in range(cfg.T):
        c = min(t + 2, cfg.W)
        gt = data["gt"][t + 2 - c: t + 2].transpose(2, 0, 1)       # [N, c, 3]
        err = gpu["poses"][t, :, :c] - gt
        err[..., 2] = np.arctan2(np.sin(err[..., 2]), np.cos(err[..., 2]))
        assert np.abs(err).max() < 2e-4 * max(1.0, np.abs(gt).max())


def _full_config(cfg, n_sample, steps=None, check_determined=False, extra_envs=(), min_determined=0.999):
    """The FULL batch in the launch configuration bench.py times (fused slam_step, default precision), compared on
    `n_sample` environments spread over the batch: newest pose (`last_pose`), covariance and ln det at every
    step, the whole window (slam_get_poses) after the last step; and, on EVERY environment, properties that hold at
    any size."""
    data = synth.generate(cfg, steps=steps)
    T = data["T"]
    envs = np.unique(np.concatenate([np.linspace(0, cfg.N - 1, n_sample), np.asarray(extra_envs, dtype=np.float64)]).astype(np.int32))
    ref = oracle.run_batch(data, cfg.iters, envs=envs)
    assert ref["bad"] == 0
    det = determined(oracle, data, cfg.iters, envs, ref) if check_determined else None
    slam = _slam(cfg.N, cfg.W, cfg.L)
    gpu = run_gpu(slam, data, cfg.iters, fused=True, want_poses=False)
    assert (gpu["status"] == 0).all()
    assert np.isfinite(gpu["cov"]).all() and np.isfinite(gpu["logdet"]).all() and np.isfinite(gpu["last_pose"]).all()
    _check(_sub(gpu, envs), ref, what=("last_pose", "cov", "logdet"), det=det, min_determined=min_determined)
    _window_after_step(slam, ref, T, envs, det)
    S = gpu["cov"]
    assert np.array_equal(S, S.transpose(0, 1, 3, 2))
    assert (np.linalg.eigvalsh(S.reshape(-1, 3, 3)).min(axis=1) > 0).all()
    return slam, data, envs, ref, gpu


def test_config1_full_size_every_env():
    _full_config(synth.CONFIGS[1], synth.CONFIGS[1].N)      # all 750 environments x 500 steps


def test_config2_full_size_sampled_envs():
    _full_config(synth.CONFIGS[2], 256)


def test_config3_full_size_sampled_envs():
    """The headline configuration: 256 environments x all 300 steps at the stated tolerances on every env-step the
    oracle determines (all but ~1e-4 of them, tests/helpers.determined); the windows fp32 cannot carry go through
    the fp64 kernel, and that really happened."""
    cfg = synth.CONFIGS[3]
    slam, data, envs, ref, gpu = _full_config(cfg, 256, check_determined=True)
    st = slam.get_stats()
    assert 0 < st["fp64_calls"] < 0.15 * cfg.N * cfg.T, st     # a few percent of the env-steps (measured: 7.7 %)
    # landmarks: the read-out against the oracle's (single environments driven step by step)
    lm, act = slam.get_landmarks()
    lm, act = lm.cpu().numpy(), act.cpu().numpy().view(np.uint32)
    for q in (0, 100, 255):
        env = int(envs[q])
        one = synth.generate(cfg, env_ids=np.array([env], np.int32))
        o = oracle.Oracle(cfg.W, cfg.L)
        drive(o, one, 0, cfg.iters)
        olm, oact = o.landmarks()
        gact = np.array([(int(act[l // 32, env]) >> (l % 32)) & 1 for l in range(cfg.L)])
        assert np.array_equal(gact, oact)
        d = np.abs(lm[:, :, env].T - olm)
        assert d.max() <= 1e-4 * max(1.0, np.abs(olm).max()), (env, d.max())


def test_config3_environments_that_come_back_from_fp64():
    """Environments that re-observe a landmark after dead reckoning (the fp64 kernel takes them), lose sight of the
    map again and dead-reckon on: found on a 4096-environment sample of config 3 as the env-steps where a hand-over
    back to fp32 by the pivot ratio alone went beyond tolerance tens of steps later (up to 2.0 x in ln det).  With
    the rule of slam_ref64_kernel -- back to fp32 only while the newest pose sees at least three landmarks -- they
    hold the stated tolerances on every env-step the oracle determines, like everybody else.  (The sample is
    hand-picked for trouble, so fewer of its env-steps are determined than of a uniform sample: measured 98.3 %.)"""
    cfg = synth.CONFIGS[3]
    found = (11512, 2132, 16216, 12552, 4140, 10608, 852, 16156, 7592, 11540, 6584, 15300)
    _full_config(cfg, 32, check_determined=True, extra_envs=found, min_determined=0.97)


@pytest.mark.parametrize("N,n_sample,steps", [(256, 64, 70), (16384, 128, None), (65536, 64, 70)])
def test_config4_sweep_sampled_envs(N, n_sample, steps):
    _full_config(synth.config4(N), n_sample, steps=steps)


def test_device_reference_agrees_at_full_batch_config3():
    """at full batch the oracle covers a sample; EVERY environment is
    diffed against the device reference (precision mode 2: the fp64 kernel, an independent second implementation
    of the same mathematics: dense packed storage, right-looking factorisation, CTA per environment).  While the
    robot is among the landmarks (steps 1..60 here) both must agree within the stated tolerances on all 16384."""
    cfg = synth.CONFIGS[3]
    data = synth.generate(cfg, steps=60)
    a = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    slam = _slam(cfg.N, cfg.W, cfg.L)
    slam.set_precision(2)
    b = run_gpu(slam, data, cfg.iters, fused=True, want_poses=False)
    assert slam.get_stats()["fp64_calls"] == cfg.N * 61       # observe_first + 60 steps, every environment
    dg = np.sqrt(np.einsum("tnii->tni", b["cov"]))
    ec = (np.abs(a["cov"] - b["cov"]) / (1e-3 * dg[..., :, None] * dg[..., None, :])).max()
    el = (np.abs(a["logdet"] - b["logdet"]) / 1e-3).max()
    d = a["last_pose"] - b["last_pose"]
    d[..., 2] = np.arctan2(np.sin(d[..., 2]), np.cos(d[..., 2]))
    ep = (np.abs(d).max(axis=2) / (1e-4 * np.maximum(1.0, np.abs(b["last_pose"]).max(axis=2)))).max()
    assert max(ec, el, ep) <= 1.0, (ec, el, ep)


def test_outputs_permute_with_the_environments():
    """Environments are independent: permuting the columns of every input permutes the
    outputs bit for bit, whichever CTA, team, round or cost-order position an environment lands on."""
    cfg = synth.Config("perm", N=1500, W=12, L=6, iters=2, T=40, p_lc=0.2, seed=21)
    data = synth.generate(cfg)
    rng = np.random.default_rng(5)
    perm = rng.permutation(cfg.N)
    pd = dict(data)
    for k in ("odom", "lc_back", "lc_meas", "rb_mask", "rb_meas"):
        pd[k] = np.ascontiguousarray(data[k][..., perm])
    a = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    b = run_gpu(_slam(cfg.N, cfg.W, cfg.L), pd, cfg.iters, fused=True, want_poses=False)
    for k in ("cov", "logdet", "last_pose"):
        assert np.array_equal(a[k][:, perm], b[k]), k


def test_step_time_does_not_depend_on_the_step_index():
    """PAPER.md:144 "constant-time updates independent of trajectory length": once the window is full the
    per-step device time of a pose-only configuration (whose structure is stationary) stays flat: the mean over
    steps 150..249 and over steps 400..499 of config 2 agree within 5 %."""
    cfg = synth.CONFIGS[2]
    data = synth.generate(cfg)
    dev = to_dev(data)
    slam = _slam(cfg.N, cfg.W, cfg.L)
    cov = torch.zeros(9, cfg.N, device="cuda")
    ld = torch.zeros(cfg.N, device="cuda")
    best = None
    for rep in range(3):
        slam.reset()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(cfg.T + 1)]
        torch.cuda.synchronize()
        ev[0].record()
        for t in range(1, cfg.T + 1):
            slam.step(dev["odom"][t - 1], dev["lc_back"][t - 1], dev["lc_meas"][t - 1], iters=cfg.iters, cov=cov, logdet=ld)
            ev[t].record()
        torch.cuda.synchronize()
        ms = np.array([ev[t].elapsed_time(ev[t + 1]) for t in range(cfg.T)])
        best = ms if best is None else np.minimum(best, ms)
    early, late = best[150:250].mean(), best[400:500].mean()
    assert abs(late / early - 1.0) <= 0.05, (early, late)
    assert best[:cfg.W - 2].mean() < early        # the window-fill phase is cheaper, never dearer


def test_state_errors_and_ignored_inputs():
    from paper_2603_25834_b200.binding import SLAM_EINVAL, SLAM_ESTATE, SlamError
    N, W = 8, 4
    slam = _slam(N, W, 0)
    z = torch.zeros(3, N, device="cuda")
    z[0] = 0.1
    with pytest.raises(SlamError) as e:
        slam.marginalize_oldest()
    assert e.value.code == SLAM_ESTATE
    assert slam.count == 1
    prior = slam.marginal_cov().cpu().numpy().reshape(3, 3, N)[:, :, 0]   # count == 1: the prior covariance
    assert np.allclose(np.diag(prior), np.array(synth.PRIOR_SIGMA) ** 2, rtol=1e-5)
    # a loop closure whose target already left the window is ignored, not an error
    back = torch.full((N,), 40, dtype=torch.int32, device="cuda")
    slam.push_step(z, back, z)
    slam.push_step(z)
    slam.push_step(z)
    assert slam.count == W
    with pytest.raises(SlamError) as e:
        slam.push_step(z)
    assert e.value.code == SLAM_ESTATE
    with pytest.raises(SlamError) as e:
        slam.solve(-1)
    assert e.value.code == SLAM_EINVAL
    with pytest.raises(SlamError):
        slam.push_step(z.cpu())
    slam.solve(0)
    slam.solve(2)
    ld, dopt = slam.dopt()
    assert np.allclose(np.exp(ld.cpu().numpy() / 3), dopt.cpu().numpy(), rtol=1e-5)
    # pure odometry chain: equals a chain without the ignored loop closure
    ref = _slam(N, W, 0)
    for _ in range(3):
        ref.push_step(z)
    ref.solve(2)
    assert torch.equal(ref.dopt()[0], ld)
    assert (slam.get_status() == 0).all()
    slam.reset()
    assert slam.count == 1


def test_not_pd_is_flagged_not_fatal():
    # a landmark at (numerically) zero range makes the bearing Jacobian blow up: flagged, no crash
    N, W, L = 4, 4, 1
    slam = _slam(N, W, L)
    mask = torch.ones(1, N, dtype=torch.int32, device="cuda")
    meas = torch.zeros(2, L, N, device="cuda")
    slam.observe_first(mask, meas)
    z = torch.zeros(3, N, device="cuda")
    slam.push_step(z, None, None, mask, meas)
    slam.solve(2)
    slam.marginal_cov()
    st = slam.get_status().cpu().numpy()
    assert (st != 0).all()


def test_step_host_matches_device_step():
    cfg = synth.Config("h", N=50, W=6, L=5, iters=2, T=20, p_lc=0.3, seed=2)
    data = synth.generate(cfg)
    a = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    slam = _slam(cfg.N, cfg.W, cfg.L)
    dev = to_dev(data)
    slam.reset()
    slam.observe_first(dev["rb_mask"][0], dev["rb_meas"][0])
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    cov = torch.zeros(9, cfg.N).pin_memory()
    ld = torch.zeros(cfg.N).pin_memory()
    for t in range(1, cfg.T + 1):
        slam.step_host(pin(data["odom"][t - 1]), pin(data["lc_back"][t - 1]), pin(data["lc_meas"][t - 1]),
                       pin(data["rb_mask"][t].view(np.int32)), pin(data["rb_meas"][t]), iters=cfg.iters, cov=cov, logdet=ld)
        torch.cuda.synchronize()
        assert np.array_equal(ld.numpy().astype(np.float64), a["logdet"][t - 1])


def test_results_do_not_depend_on_capacity_or_team(monkeypatch):
    """The size of the shared-memory pool only decides in WHICH round of its CTA an environment is solved
    (one that does not fit waits and goes first in the next round); the arithmetic is the same, so outputs
    are bit-equal.  Different team sizes change summation order in a few reductions: equal within the
    tolerances."""
    cfg = synth.Config("cap", N=200, W=40, L=0, iters=3, T=70, p_lc=0.3, seed=11)
    data = synth.generate(cfg)
    monkeypatch.setenv("SLAM_POOL_FRAC", "1.0")
    monkeypatch.setenv("SLAM_MAX_WPC", "2")               # a pool with room for every team
    slam = _slam(cfg.N, cfg.W, cfg.L)
    a = run_gpu(slam, data, cfg.iters, fused=True, want_poses=False)
    assert slam.get_stats()["waited"] == 0
    monkeypatch.delenv("SLAM_MAX_WPC")
    monkeypatch.setenv("SLAM_POOL_FRAC", "0.01")          # clamped to the dense need of ONE environment
    slam = _slam(cfg.N, cfg.W, cfg.L)
    b = run_gpu(slam, data, cfg.iters, fused=True, want_poses=False)
    st = slam.get_stats()
    assert st["waited"] > 0, st                           # teams really waited for pool space
    assert np.array_equal(a["cov"], b["cov"]) and np.array_equal(a["logdet"], b["logdet"])
    assert (b["status"] == 0).all()
    monkeypatch.delenv("SLAM_POOL_FRAC")
    monkeypatch.setenv("SLAM_PREFETCH", "1")              # the L2 bulk prefetch of the next round's records is a hint only
    p0 = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(a["cov"], p0["cov"]) and np.array_equal(a["logdet"], p0["logdet"])
    monkeypatch.delenv("SLAM_PREFETCH")
    monkeypatch.setenv("SLAM_DYNQ", "0")                  # static deal of the list to the CTAs instead of the one queue
    q0 = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(a["cov"], q0["cov"]) and np.array_equal(a["logdet"], q0["logdet"])
    monkeypatch.delenv("SLAM_DYNQ")
    ref = oracle.run_batch(data, cfg.iters, envs=np.arange(0, cfg.N, 25, dtype=np.int32))
    for team in ("32", "128"):
        monkeypatch.setenv("SLAM_TEAM", team)
        c = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
        _check(_sub(c, np.arange(0, cfg.N, 25)), ref, what=("cov", "logdet"))
    monkeypatch.delenv("SLAM_TEAM")


@pytest.mark.gpu
@pytest.mark.parametrize("W,L,p_lc,pairs", [(40, 0, 0.3, "1"), (40, 0, 0.3, "0"), (7, 9, 0.3, "1"), (64, 64, 0.1, "1")])
def test_envelope_rows_in_pairs_or_fours(monkeypatch, W, L, p_lc, pairs):
    """SLAM_PAIRS selects how the envelope rows are grouped (storage and the split dot products of the
    factorisation); both groupings hold the stated tolerances, with and without landmarks."""
    monkeypatch.setenv("SLAM_PAIRS", pairs)
    N, T = (3, 68) if W == 64 else (60, 60)
    cfg = synth.Config("pairs", N=N, W=W, L=L, iters=2, T=T, p_lc=p_lc, seed=13)
    data = synth.generate(cfg)
    ref = oracle.run_batch(data, cfg.iters)
    gpu = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref, what=("cov", "logdet"))


@pytest.mark.parametrize("W,L,p_lc", [(8, 0, 0.3), (6, 7, 0.2)])
def test_unary_pose_factor_next1(W, L, p_lc):
    """NEXT-1: unary absolute-pose factors with caller-supplied information."""
    cfg = synth.Config("un", N=40, W=W, L=L, iters=2, T=50, p_lc=p_lc, seed=17, p_unary=0.4)
    data = synth.generate(cfg)
    ref = oracle.run_batch(data, cfg.iters)
    assert ref["bad"] == 0
    gpu = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref)
    _fused_equals_separate(cfg, data, ref)
    # the absolute measurements really bound the uncertainty: without them log-det keeps growing
    plain = synth.generate(synth.Config("pl", N=40, W=W, L=L, iters=2, T=50, p_lc=p_lc, seed=17))
    ref_plain = oracle.run_batch(plain, cfg.iters, want=("logdet",))
    assert ref["logdet"][-1].mean() < ref_plain["logdet"][-1].mean() - 1.0


@pytest.mark.parametrize("W,L,p_lc", [(7, 0, 0.3), (6, 6, 0.2)])
def test_per_env_reset_next2(W, L, p_lc):
    """NEXT-2: slam_reset_envs restarts single environments mid-run while the others keep their windows."""
    cfg = synth.Config("rs", N=60, W=W, L=L, iters=2, T=70, p_lc=p_lc, seed=23, p_reset=0.05, p_unary=0.1)
    data = synth.generate(cfg)
    assert data["reset"].sum() > 50
    ref = oracle.run_batch(data, cfg.iters)
    assert ref["bad"] == 0
    gpu = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref)
    _fused_equals_separate(cfg, data, ref)
