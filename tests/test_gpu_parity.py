"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on identical seeded inputs.

Tolerances are BASELINE.json north_star's, in the reading R23 of DESIGN.md (written in
tests/gpu_driver.parity_errors): poses rel 1e-4, covariance 1e-3 of sqrt(S_ii S_jj), ln det abs 1e-3.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2603_25834_b200 import synth
from tests.gpu_driver import parity_errors, run_gpu, to_dev

pytestmark = pytest.mark.gpu


def _slam(N, W, L):
    from paper_2603_25834_b200.binding import FixedLagSlam
    return FixedLagSlam(N, W, L)


PROBE_FORK = 1.0 / 12.0        # an environment "forks" when fp32 STORAGE alone costs 1/12 of a tolerance
FORKED_FACTOR = 100.0          # after the fork (loose sanity bound): error <= 100 x max(1, probe's running maximum)
MAX_EXCEED_FRACTION = 0.01     # at most 1 % of all env-steps may exceed the stated tolerance at all
MIN_STRICT_COVERAGE = 0.80


def _check(gpu, ref, what=("poses", "cov", "logdet"), probe=None, min_coverage=MIN_STRICT_COVERAGE):
    """Every (step, env) must be within the stated tolerances R23 (error <= 1.0 in tolerance units).

    Conditioning: in config 3, late in the run, the information matrix of some
    environments is so ill-conditioned that the ORACLE's own outputs move by a tolerance or more when H,
    b, the prior and the state are merely rounded to fp32 (`probe` = that run of the same fp64 algorithm).
    No fp32 implementation can follow the oracle there, and the two trajectories stay apart afterwards
    (the prior is linearised at different points).  So: an environment is held to the STATED tolerance
    on every step before the first one where the probe's error reaches 1/12 of a tolerance (its "fork");
    after the fork the two runs are different trajectories (chaotic sensitivity), so only a loose sanity
    bound applies (100 x max(1, the probe's running maximum)); and over everything at most 1 % of env-steps
    may exceed the stated tolerance.  Pose-only configs never fork."""
    err = parity_errors(gpu, ref)
    keys = [k for k in what if k in err]
    assert keys
    G = np.max([err[k] for k in keys], axis=0)
    assert np.isfinite(G).all()
    if probe is None:
        worst = float(G.max())
        assert worst <= 1.0, f"{worst:.3g} x tolerance at {np.unravel_index(G.argmax(), G.shape)}"
        return err
    perr = parity_errors(probe, ref)
    P = np.max([perr[k] for k in keys], axis=0)
    T = G.shape[0]
    forked = np.maximum.accumulate(P > PROBE_FORK, axis=0)
    strict = ~forked
    assert strict.mean() >= min_coverage, f"strict coverage {strict.mean():.3f}"
    if strict.any():
        worst = float(G[strict].max())
        assert worst <= 1.0, f"{worst:.3g} x tolerance on a well-conditioned env-step"
    bound = FORKED_FACTOR * np.maximum(1.0, np.maximum.accumulate(P, axis=0))
    assert (G <= bound).all(), f"forked env-step beyond {FORKED_FACTOR} x probe: {float((G / bound).max()):.3g}"
    assert (G > 1.0).mean() <= MAX_EXCEED_FRACTION, f"{(G > 1.0).mean():.3%} of env-steps exceed the stated tolerance"
    return err


def _sub(gpu, envs):
    return {k: (v[:, envs] if k != "status" else v[envs]) for k, v in gpu.items()}


def test_config0_all_envs_all_steps():
    cfg = synth.CONFIGS[0]
    data = synth.generate(cfg)
    ref = oracle.run_batch(data, cfg.iters)
    gpu = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=False)
    assert (gpu["status"] == 0).all()
    _check(gpu, ref)
    fused = run_gpu(_slam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)
    _check(fused, ref, what=("cov", "logdet"))


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
    a = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=False, want_poses=False)
    b = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(a["cov"], b["cov"])
    assert np.array_equal(a["logdet"], b["logdet"])
    # and the run is reproducible launch to launch
    c = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(b["cov"], c["cov"])


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


def _full_config(cfg, n_sample, steps=None):
    data = synth.generate(cfg, steps=steps)
    envs = np.unique(np.linspace(0, cfg.N - 1, n_sample).astype(np.int32))
    ref = oracle.run_batch(data, cfg.iters, envs=envs)
    probe = oracle.run_batch(data, cfg.iters, envs=envs, f32_storage=True)
    assert ref["bad"] == 0
    slam = _slam(cfg.N, cfg.W, cfg.L)
    gpu = run_gpu(slam, data, cfg.iters, fused=True, want_poses=False)   # the launch configuration bench.py times
    assert (gpu["status"] == 0).all()
    assert np.isfinite(gpu["cov"]).all() and np.isfinite(gpu["logdet"]).all()
    _check(_sub(gpu, envs), ref, what=("cov", "logdet"), probe=probe)
    # properties that hold at any size: symmetric positive-definite covariances on EVERY env and step
    S = gpu["cov"]
    assert np.array_equal(S, S.transpose(0, 1, 3, 2))
    assert (np.linalg.eigvalsh(S.reshape(-1, 3, 3)).min(axis=1) > 0).all()
    return data, envs, ref, probe


def test_config1_full_size_sampled_envs():
    cfg = synth.CONFIGS[1]
    data, envs, ref, probe = _full_config(cfg, 24)
    # poses through the separate calls on the same sampled environments
    sub = synth.generate(cfg, env_ids=envs)
    gpu = run_gpu(_slam(len(envs), cfg.W, cfg.L), sub, cfg.iters, fused=False)
    _check(gpu, ref, probe=probe, min_coverage=1.0)      # pose-only: no environment forks


def test_config2_full_size_sampled_envs():
    _full_config(synth.CONFIGS[2], 10)


def test_config3_full_size_sampled_envs():
    cfg = synth.CONFIGS[3]
    data, envs, ref, probe = _full_config(cfg, 48)
    sub = synth.generate(cfg, env_ids=envs)
    gpu = run_gpu(_slam(len(envs), cfg.W, cfg.L), sub, cfg.iters, fused=False)
    _check(gpu, ref, probe=probe)


def test_config4_n16384_sampled_envs():
    _full_config(synth.config4(16384), 6)


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
    fused = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(fused["cov"], gpu["cov"]) and np.array_equal(fused["logdet"], gpu["logdet"])
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
    fused = run_gpu(_slam(cfg.N, W, L), data, cfg.iters, fused=True, want_poses=False)
    assert np.array_equal(fused["cov"], gpu["cov"]) and np.array_equal(fused["logdet"], gpu["logdet"])
