"""Writes chain_logdet.txt from the closed form alone (no oracle, no CUDA code).

Pure-translation odometry chain, step d along x, heading 0, prior variances P0, odometry variances
Q (BASELINE.json sigmas).  The newest pose's marginal covariance after k steps (eq. (6) of the paper,
PAPER.md:158-163, read as the last block of the inverse, R14) is the k-fold EKF prediction
    S_xx = p_x + k q_x
    S_yy = p_y + k^2 d^2 p_t + k q_y + d^2 q_t (k-1)k(2k-1)/6
    S_yt = k d p_t + d q_t k(k-1)/2
    S_tt = p_t + k q_t
"""
import math
import os

P0 = (0.01 ** 2, 0.01 ** 2, 0.005 ** 2)
Q = (0.05 ** 2, 0.05 ** 2, 0.02 ** 2)
D = 0.2


def logdet(k):
    sxx = P0[0] + k * Q[0]
    syy = P0[1] + k * k * D * D * P0[2] + k * Q[1] + D * D * Q[2] * (k - 1) * k * (2 * k - 1) / 6.0
    syt = k * D * P0[2] + D * Q[2] * k * (k - 1) / 2.0
    stt = P0[2] + k * Q[2]
    return math.log(sxx * (syy * stt - syt * syt))


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "chain_logdet.txt")
    with open(path, "w") as f:
        f.write("# ln det Sigma_k of the newest pose on a pure-translation chain (d=0.2 m, BASELINE.json sigmas).\n")
        f.write("# Source: closed form in make_chain_logdet.py (paper eq. (6), PAPER.md:158-163; the paper prints\n")
        f.write("# no numeric example).  SURVEY.md 8(c) quotes k=1,2,5,10,40: -19.667547 -17.655162 -14.936988\n")
        f.write("# -12.832615 -8.118278.\n# k  lndet\n")
        for k in (1, 2, 5, 10, 20, 40):
            f.write(f"{k} {logdet(k):.9f}\n")
