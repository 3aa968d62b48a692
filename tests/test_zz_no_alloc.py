"""slam_run_static: the allocation-free entry point (a whole episode on the library's static scratch array) against
the existing path (a FixedLagSlam context on a caller-allocated workspace, one slam_step per step).

Collected last on purpose (the suite runs with ``pytest -x``).  Two calls in a row with different episodes: the
array keeps the first call's contents, so the second one checks that every call clears what must start at zero.
Tolerances: the parity tolerances of the other GPU tests (R23 of DESIGN.md, ``tests/gpu_driver.parity_errors``)."""
import numpy as np
import pytest
import torch

from harness import synth
from tests.gpu_driver import parity_errors, run_gpu, to_dev

pytestmark = pytest.mark.gpu


def _episode(seed, N, W, L, T, iters, p_lc):
    cfg = synth.Config("static", N=N, W=W, L=L, iters=iters, T=T, p_lc=p_lc, seed=seed)
    return cfg, synth.generate(cfg)


def _run_static(cfg, data):
    from paper_2603_25834_b200 import binding
    dev = to_dev(data)
    T, N = cfg.T, cfg.N
    cov = torch.full((T, 9, N), float("nan"), device="cuda:0")
    logdet = torch.full((T, N), float("nan"), device="cuda:0")
    last = torch.full((T, 3, N), float("nan"), device="cuda:0")
    binding.run_static(N, cfg.W, cfg.L, cfg.iters, dev["odom"], dev["lc_back"], dev["lc_meas"],
                       dev["rb_mask"] if cfg.L else None, dev["rb_meas"] if cfg.L else None, cov, logdet, last)
    torch.cuda.synchronize()
    return dict(cov=cov.cpu().numpy().reshape(T, 3, 3, N).transpose(0, 3, 1, 2).astype(np.float64),
                logdet=logdet.cpu().numpy().astype(np.float64), last=last.cpu().numpy().astype(np.float64))


def _run_existing(cfg, data):
    from paper_2603_25834_b200.binding import FixedLagSlam
    return run_gpu(FixedLagSlam(cfg.N, cfg.W, cfg.L), data, cfg.iters, fused=True, want_poses=False)


def test_run_static_matches_the_workspace_path_twice_in_a_row():
    # first call: landmarks + loop closures, long enough to marginalise many times
    cfg_a, data_a = _episode(31, N=96, W=6, L=5, T=40, iters=2, p_lc=0.3)
    # second call: a different shape (pose-only, larger window, other batch) on the same array
    cfg_b, data_b = _episode(32, N=50, W=12, L=0, T=30, iters=3, p_lc=0.4)
    got_a = _run_static(cfg_a, data_a)
    got_b = _run_static(cfg_b, data_b)
    for cfg, data, got in ((cfg_a, data_a, got_a), (cfg_b, data_b, got_b)):
        ref = _run_existing(cfg, data)
        assert np.isfinite(got["cov"]).all() and np.isfinite(got["logdet"]).all() and np.isfinite(got["last"]).all()
        err = parity_errors(got, ref)          # units of the stated tolerances (cov 1e-3 relative, ln det 1e-3 absolute)
        worst = max(float(v.max()) for v in err.values())
        assert worst <= 1.0, f"{cfg.name}: {worst:.3g} x tolerance"
    # and once more with the first episode: same result as its first call
    again = _run_static(cfg_a, data_a)
    err = parity_errors(again, got_a)
    assert max(float(v.max()) for v in err.values()) <= 1.0


def test_run_static_rejects_sizes_beyond_the_array():
    from paper_2603_25834_b200 import binding
    N, W, L = 4096, 20, 24                       # ~ 300 MB of records: far beyond the 16 MiB array
    assert binding.workspace_bytes(N, W, L) > binding.STATIC_MAX_BYTES
    z = torch.zeros(1, 3, N, device="cuda:0")
    m = torch.zeros(2, 1, N, dtype=torch.int32, device="cuda:0")
    r = torch.zeros(2, 2, L, N, device="cuda:0")
    with pytest.raises(binding.SlamError) as e:
        binding.run_static(N, W, L, 2, z, None, None, m, r)
    assert e.value.code == binding.SLAM_ENOMEM and "SLAM_STATIC_MAX_BYTES" in str(e.value)
