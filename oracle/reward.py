"""fp64 ORACLE of the paper's reward, eqs. (7)-(17) -- TEST INFRASTRUCTURE ONLY.

The reward is an exact closed form, so the oracle is that definition written out equation by equation
in numpy float64, in the paper's order and notation.  Hyper-parameters (lambda_*, U_hi, kappa, d_crash,
d_full) are on the paper's project page, not in the paper: they are inputs.  Pins: tests/test_reward.py
(collision case, gating limits, sign rule of eq. (17), a hand-worked example).
"""
import numpy as np


def reward(U, U_prev, dcells, d_min, collision, *, lambda_col, lambda_explore, lambda_abs, lambda_delta, u_hi, kappa,
           d_crash, d_full):
    U, U_prev, dcells, d_min = (np.asarray(x, np.float64) for x in (U, U_prev, dcells, d_min))
    collision = np.asarray(collision) != 0
    c_prev = np.clip((u_hi - U_prev) / u_hi, 0.0, 1.0) ** 2                        # (11)
    iota = np.clip(np.maximum(U_prev - U, 0.0) / kappa, 0.0, 1.0)                  # (12)
    I = c_prev + (1.0 - c_prev) * iota                                             # (10)
    R_explore = lambda_explore * dcells * I                                        # (8)
    R_abs = lambda_abs * np.exp(U_prev) * U_prev                                   # (13)
    R_delta = lambda_delta * np.exp(U_prev) * (U_prev - U)                         # (14)
    alpha_hug = np.clip((d_min - d_crash) / (d_full - d_crash), 0.0, 1.0)          # (15)
    R_explore_s = R_explore * alpha_hug                                            # (16)
    R_delta_s = np.where(U_prev - U > 0, R_delta * alpha_hug, R_delta)             # (17)
    return np.where(collision, -lambda_col, R_explore_s - R_abs + R_delta_s)       # (7)


def delta_cells(t_since_visit, T_episode, new_cell):
    """Eq. (9): 1 for a new cell, else half the fraction of the episode since the last visit."""
    t_since_visit = np.asarray(t_since_visit, np.float64)
    return np.where(np.asarray(new_cell) != 0, 1.0, 0.5 * t_since_visit / T_episode)
