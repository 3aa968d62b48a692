"""NEXT-4: reward of eqs. (7)-(17): pins of the oracle (no GPU) and GPU parity."""
import math

import numpy as np
import pytest

from oracle import reward as orw

HP = dict(lambda_col=10.0, lambda_explore=2.0, lambda_abs=0.1, lambda_delta=1.0, u_hi=2.0, kappa=1.0, d_crash=0.1, d_full=0.5)


def test_hand_worked_example():
    # U_hi = 2, U_{t-1} = 1, U_t = 0.5, kappa = 1:
    #   c = ((2 - 1) / 2)^2 = 0.25                                   (11)
    #   iota = clip(0.5 / 1) = 0.5                                   (12)
    #   I = 0.25 + 0.75 * 0.5 = 0.625                                (10)
    #   R_explore = 2 * 1 * 0.625 = 1.25                             (8)
    #   alpha = (0.3 - 0.1) / (0.5 - 0.1) = 0.5                      (15)  -> R*_explore = 0.625   (16)
    #   R_abs = 0.1 * e * 1                                          (13)
    #   R_delta = 1 * e * 0.5 > 0 -> R*_delta = 0.25 e               (17)
    #   R = 0.625 - 0.1 e + 0.25 e = 0.625 + 0.15 e                  (7)
    r = orw.reward(0.5, 1.0, 1.0, 0.3, 0, **HP)
    assert abs(float(r) - (0.625 + 0.15 * math.e)) < 1e-14


def test_collision_and_limits():
    assert float(orw.reward(0.5, 1.0, 1.0, 0.3, 1, **HP)) == -10.0                           # (7)
    # no uncertainty at t-1 and no change: c = 1, I = 1, R_abs = R_delta = 0; far from walls alpha = 1
    assert abs(float(orw.reward(0.0, 0.0, 0.7, 5.0, 0, **HP)) - 2.0 * 0.7) < 1e-15
    # at or beyond U_hi exploration pays only through the information gain iota (c = 0)
    r_hi = orw.reward(3.0, 3.0, 1.0, 5.0, 0, **HP)
    assert abs(float(r_hi) - (-0.1 * math.exp(3.0) * 3.0)) < 1e-12
    # iota saturates at a drop of kappa
    a = orw.reward(1.0, 2.5, 1.0, 5.0, 0, **HP) - orw.reward(1.0, 2.5, 0.0, 5.0, 0, **HP)
    assert abs(float(a) - 2.0) < 1e-12
    # eq. (17): a negative differential term is NOT weakened near a wall, a positive one is
    near, far = dict(d_min=0.1), dict(d_min=5.0)
    worse = [float(orw.reward(1.5, 1.0, 0.0, dm, 0, **HP)) for dm in (0.1, 5.0)]
    assert worse[0] == worse[1]
    better = [float(orw.reward(0.5, 1.0, 0.0, dm, 0, **HP)) for dm in (0.1, 5.0)]
    assert better[0] < better[1] and abs(better[0] - (-0.1 * math.e)) < 1e-14
    # eq. (9)
    assert float(orw.delta_cells(0, 2048, 1)) == 1.0 and float(orw.delta_cells(2048, 2048, 0)) == 0.5


def test_monotone_in_uncertainty_reduction():
    U = np.linspace(0.0, 1.0, 21)
    r = orw.reward(U, 1.0, 1.0, 5.0, 0, **HP)
    assert (np.diff(r) < 0).all()       # the more uncertainty is left, the smaller the reward


@pytest.mark.gpu
def test_reward_kernel_matches_oracle():
    import torch
    from paper_2603_25834_b200.binding import FixedLagSlam, RewardParams
    N = 1000
    rng = np.random.default_rng(0)
    U, Up = rng.uniform(0, 3, N), rng.uniform(0, 3, N)
    dc, dm = rng.uniform(0, 1, N), rng.uniform(0, 1, N)
    col = (rng.uniform(size=N) < 0.1).astype(np.int32)
    slam = FixedLagSlam(N, 4, 0)
    f = lambda x: torch.from_numpy(np.asarray(x, np.float32)).cuda()
    p = RewardParams(**{k: float(v) for k, v in HP.items()})
    out = slam.reward(p, f(U), f(Up), f(dc), f(dm), torch.from_numpy(col).cuda()).cpu().numpy().astype(np.float64)
    ref = orw.reward(f(U).cpu().numpy(), f(Up).cpu().numpy(), f(dc).cpu().numpy(), f(dm).cpu().numpy(), col, **HP)
    assert np.allclose(out, ref, rtol=2e-6, atol=1e-6)
