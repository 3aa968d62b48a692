"""Seeded synthetic multi-robot trajectories: the stand-in for the paper's simulator.

The paper measures only inside Isaac Sim / Isaac Lab, which is not available;
BASELINE.json replaces it by synthetic SE(2) trajectories with the factor sets and noise levels of
its ``configs``.  This module draws those inputs.  It is HARNESS code used
by the tests, ``bench.py`` and ``__graft_entry__.smoke()`` to feed BOTH the CUDA library and the fp64
oracle the same arrays.  It holds none of the method's arithmetic (no residuals, Jacobians,
Hessians, solves): only the ground-truth motion model needed to simulate measurements.

Layout of every array is "environment fastest" (``[..., N]``), matching ``include/slam.h``.

Random numbers: one ``splitmix64`` stream per environment, seeded from ``(seed, env)``; uniforms from
the top 53 bits; normals by Box-Muller (cosine branch, two uniforms per normal).  The draw order per
environment and step is fixed (see :func:`generate`), so a trajectory of environment ``i`` does not
depend on ``N`` and the noise-free variant (``noise_scale=0``) follows the same ground truth.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_TWO_PI = 2.0 * math.pi


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json workload (``configs[k]``)."""

    name: str
    N: int          # environments
    W: int          # window (poses)
    L: int          # landmarks per environment
    iters: int      # Gauss-Newton iterations per step
    T: int          # environment steps
    p_lc: float     # loop-closure probability per step
    seed: int = 0
    p_unary: float = 0.0   # NEXT-1: probability of a scan-match style absolute-pose measurement per step
    p_reset: float = 0.0   # NEXT-2: probability of an episode reset (SLAM restarts at the true pose) per step


# BASELINE.json `configs`, in order.  Config 4 is a sweep over N; `config4(N)` builds one point.
CONFIGS = {
    0: Config("cfg0_pose_only", N=4, W=10, L=0, iters=3, T=100, p_lc=0.0),
    1: Config("cfg1_loops_750", N=750, W=20, L=0, iters=3, T=500, p_lc=0.1),
    2: Config("cfg2_loops_4096", N=4096, W=30, L=0, iters=3, T=500, p_lc=0.2),
    3: Config("cfg3_landmarks_16384", N=16384, W=20, L=24, iters=2, T=300, p_lc=0.0),
}
CONFIG4_NS = (256, 1024, 4096, 16384, 65536)


def config4(N: int) -> Config:
    return Config(f"cfg4_stress_{N}", N=N, W=50, L=0, iters=3, T=200, p_lc=0.2)


# Noise levels of BASELINE.json (sigma): these are also the library defaults in include/slam.h.
PRIOR_SIGMA = (0.01, 0.01, 0.005)
ODO_SIGMA = (0.05, 0.05, 0.02)
LC_SIGMA = (0.10, 0.10, 0.03)
RB_SIGMA = (0.05, 0.01)
UNARY_SIGMA = (0.03, 0.03, 0.01)   # absolute-pose measurement noise in the robot frame at match score 1
RB_MIN_RANGE = 0.5
RB_MAX_RANGE = 8.0
LM_BOX_HALF = 10.0


class _Streams:
    """N independent splitmix64 streams advanced in lock-step (vectorised over environments)."""

    def __init__(self, seed: int, env_ids: np.ndarray):
        with np.errstate(over="ignore"):
            s = np.uint64(seed) * _GOLDEN + env_ids.astype(np.uint64) * np.uint64(0xD1B54A32D192ED03)
            self.state = s
            # one scrambling round so that neighbouring environments start far apart
            self.state = self._next_u64()

    def _next_u64(self) -> np.ndarray:
        with np.errstate(over="ignore"):
            self.state = self.state + _GOLDEN
            z = self.state.copy()
            z = (z ^ (z >> np.uint64(30))) * _M1
            z = (z ^ (z >> np.uint64(27))) * _M2
            z = z ^ (z >> np.uint64(31))
        return z

    def uniform(self) -> np.ndarray:
        """U[0,1) with 53 random bits."""
        return (self._next_u64() >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)

    def normal(self) -> np.ndarray:
        """N(0,1): Box-Muller, cosine branch; consumes two uniforms."""
        u1 = self.uniform()
        u2 = self.uniform()
        return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(_TWO_PI * u2)


def wrap(x):
    """Wrap an angle to (-pi, pi]."""
    return np.arctan2(np.sin(x), np.cos(x))


def compose(p, u):
    """Ground-truth motion model p (+) u on SE(2); p, u are [3, N]."""
    c, s = np.cos(p[2]), np.sin(p[2])
    return np.stack([p[0] + c * u[0] - s * u[1], p[1] + s * u[0] + c * u[1], wrap(p[2] + u[2])])


def between(p, q):
    """Pose q expressed in the frame of pose p (both [3, N])."""
    c, s = np.cos(p[2]), np.sin(p[2])
    dx, dy = q[0] - p[0], q[1] - p[1]
    return np.stack([c * dx + s * dy, -s * dx + c * dy, wrap(q[2] - p[2])])


def generate(cfg: Config, *, noise_scale: float = 1.0, dtype=np.float32, env_ids=None,
             steps: int | None = None) -> dict:
    """Draw all inputs of one workload.

    Per environment: ``GT_0 = (0,0,0)``; if ``L > 0`` the landmark map ``U([-10,10]^2)`` is drawn
    first (x then y per landmark), then the range-bearing observation from ``GT_0`` (two normals per
    landmark, always drawn).  For step t = 1..T in this order:

    1. true motion ``u = (U(0,0.3), N(0,0.02^2), U(-0.3,0.3))``; ``GT_t = GT_{t-1} (+) u``
    2. ``odom = u + noise_scale * N(0, diag(0.05^2, 0.05^2, 0.02^2))``
    3. ``q ~ U(0,1)``, ``age ~ U{1..min(t, W-1)}``, three normals (always drawn); a loop closure to
       the pose ``age`` steps older is emitted iff ``q < p_lc``
    4. for each landmark: two normals (always drawn); visible iff ``0.5 <= range_GT <= 8``

    Returns a dict of arrays, environment index last:
      ``odom[T,3,N]``, ``lc_back[T,N]`` (int32, 0 = none), ``lc_meas[T,3,N]``,
      ``rb_mask[T+1,ceil(L/32),N]`` (uint32), ``rb_meas[T+1,2,L,N]`` (range, bearing),
      ``gt[T+1,3,N]`` and ``lm[2,L,N]`` (float64, for tests only).
    Measurement arrays have ``dtype`` (float32 = what the library consumes; float64 for oracle pins).
    """
    W, L = cfg.W, cfg.L
    T = cfg.T if steps is None else int(steps)
    if env_ids is None:
        env_ids = np.arange(cfg.N, dtype=np.int64)
    env_ids = np.asarray(env_ids, dtype=np.int64)
    N = env_ids.shape[0]
    rng = _Streams(cfg.seed, env_ids)
    ns = float(noise_scale)
    nwords = (L + 31) // 32

    odom = np.zeros((T, 3, N), dtype)
    lc_back = np.zeros((T, N), np.int32)
    lc_meas = np.zeros((T, 3, N), dtype)
    rb_mask = np.zeros((T + 1, nwords, N), np.uint32)
    rb_meas = np.zeros((T + 1, 2, L, N), dtype)
    gt = np.zeros((T + 1, 3, N), np.float64)
    lm = np.zeros((2, L, N), np.float64)
    un_valid = np.zeros((T, N), np.int32) if cfg.p_unary > 0 else None
    un_pose = np.zeros((T, 3, N), dtype) if cfg.p_unary > 0 else None
    un_info = np.zeros((T, 6, N), dtype) if cfg.p_unary > 0 else None
    reset = np.zeros((T, N), np.int32) if cfg.p_reset > 0 else None
    reset_pose = np.zeros((T, 3, N), dtype) if cfg.p_reset > 0 else None

    for l in range(L):
        lm[0, l] = (2.0 * rng.uniform() - 1.0) * LM_BOX_HALF
        lm[1, l] = (2.0 * rng.uniform() - 1.0) * LM_BOX_HALF

    def observe(t: int, pose: np.ndarray) -> None:
        for l in range(L):
            dx, dy = lm[0, l] - pose[0], lm[1, l] - pose[1]
            rho = np.hypot(dx, dy)
            beta = wrap(np.arctan2(dy, dx) - pose[2])
            n_r = rng.normal()
            n_b = rng.normal()
            vis = (rho >= RB_MIN_RANGE) & (rho <= RB_MAX_RANGE)
            rb_meas[t, 0, l] = np.where(vis, rho + ns * RB_SIGMA[0] * n_r, 0.0)
            rb_meas[t, 1, l] = np.where(vis, wrap(beta + ns * RB_SIGMA[1] * n_b), 0.0)
            rb_mask[t, l // 32] |= (vis.astype(np.uint32) << np.uint32(l % 32))

    if L > 0:
        observe(0, gt[0])

    for t in range(1, T + 1):
        u = np.stack([0.3 * rng.uniform(), 0.02 * rng.normal(), 0.6 * rng.uniform() - 0.3])
        gt[t] = compose(gt[t - 1], u)
        for k in range(3):
            odom[t - 1, k] = u[k] + ns * ODO_SIGMA[k] * rng.normal()
        q = rng.uniform()
        c_old = min(t, W - 1)
        age = 1 + np.minimum((rng.uniform() * c_old).astype(np.int64), c_old - 1)
        noise = [rng.normal() for _ in range(3)]
        has = q < cfg.p_lc
        if has.any():
            # ground-truth pose `age` steps older, per environment
            tgt = np.take_along_axis(gt[: t + 1], (t - age)[None, None, :].repeat(3, 1), axis=0)[0]
            z = between(tgt, gt[t])
            z = np.stack([z[0] + ns * LC_SIGMA[0] * noise[0], z[1] + ns * LC_SIGMA[1] * noise[1],
                          wrap(z[2] + ns * LC_SIGMA[2] * noise[2])])
            lc_back[t - 1] = np.where(has, age, 0).astype(np.int32)
            lc_meas[t - 1] = np.where(has[None, :], z, 0.0)
        if L > 0:
            observe(t, gt[t])
        if cfg.p_unary > 0:
            # 5. (only when p_unary > 0, drawn last so that the other streams are unchanged): q ~ U(0,1),
            #    match score ~ U(0.3,1), three normals; measurement = GT_t + Rot(theta) * noise / sqrt(score);
            #    information = score * R diag(1/sigma^2) R' in GLOBAL coordinates, packed (xx, xy, yy, xt, yt, tt)
            q = rng.uniform()
            score = 0.3 + 0.7 * rng.uniform()
            nz = [rng.normal() for _ in range(3)]
            has = q < cfg.p_unary
            c, s_ = np.cos(gt[t, 2]), np.sin(gt[t, 2])
            ex = ns * UNARY_SIGMA[0] * nz[0] / np.sqrt(score)
            ey = ns * UNARY_SIGMA[1] * nz[1] / np.sqrt(score)
            et = ns * UNARY_SIGMA[2] * nz[2] / np.sqrt(score)
            zu = np.stack([gt[t, 0] + c * ex - s_ * ey, gt[t, 1] + s_ * ex + c * ey, wrap(gt[t, 2] + et)])
            wx, wy, wt = score / UNARY_SIGMA[0] ** 2, score / UNARY_SIGMA[1] ** 2, score / UNARY_SIGMA[2] ** 2
            info = np.stack([c * c * wx + s_ * s_ * wy, c * s_ * (wx - wy), s_ * s_ * wx + c * c * wy,
                             np.zeros_like(c), np.zeros_like(c), wt])
            un_valid[t - 1] = has.astype(np.int32)
            un_pose[t - 1] = np.where(has[None, :], zu, 0.0)
            un_info[t - 1] = np.where(has[None, :], info, 0.0)

        if cfg.p_reset > 0:
            # 6. (only when p_reset > 0, drawn last): the estimator of this environment restarts BEFORE the
            #    push of step t at the true pose GT_{t-1} (a new episode); not on the first two steps
            q = rng.uniform()
            has = (q < cfg.p_reset) & (t > 2)
            reset[t - 1] = has.astype(np.int32)
            reset_pose[t - 1] = np.where(has[None, :], gt[t - 1], 0.0)

    return dict(reset=reset, reset_pose=reset_pose, un_valid=un_valid, un_pose=un_pose, un_info=un_info, odom=odom, lc_back=lc_back, lc_meas=lc_meas, rb_mask=rb_mask, rb_meas=rb_meas,
                gt=gt, lm=lm, env_ids=env_ids, cfg=cfg, T=T)


# ----------------------------------------------------------------------------- NEXT-3: scan-matching worlds
def generate_scan_world(N: int, G: int = 128, res: float = 0.1, R: int = 128, seed: int = 0, *,
                        offset_cells=(0, 0, 0), sth: float = 0.01, range_sigma: float = 0.0, l_hi: float = 4.0,
                        l_lo: float = 2.0, dtype=np.float32) -> dict:
    """Synthetic stand-in for the paper's LiDAR + occupancy grid.

    Per environment: a rectangular room (half sizes U(2.5,4.5) m, walls on cell CENTRES) with one
    axis-aligned box obstacle; the robot at a random pose inside; a 128-ray, 180-degree scan cast
    analytically against the walls (+ N(0, range_sigma^2)); the log-odds map rasterised from the same
    walls (+l_hi on wall cells, -l_lo inside the room, 0 outside); and a predicted pose = true pose
    MINUS `offset_cells` lattice steps (res, res, sth), so that the candidate at +offset_cells is the
    true pose.  Environment-fastest arrays: ``grid[N,G,G]``, ``ranges[R,N]``, ``pose_true[3,N]``,
    ``pose_pred[3,N]``."""
    rng = _Streams(seed ^ 0x5CA1AB1E, np.arange(N, dtype=np.int64))
    half = 0.5 * G * res

    def snap(v):      # to a cell centre
        return (np.floor(v / res) + 0.5) * res

    wx, wy = snap(2.5 + 2.0 * rng.uniform()), snap(2.5 + 2.0 * rng.uniform())          # room half sizes
    bx, by = snap(-1.5 + 3.0 * rng.uniform()), snap(0.8 + 1.2 * rng.uniform())          # box centre (in front)
    bw, bh = snap(0.3 + 0.5 * rng.uniform()), snap(0.3 + 0.5 * rng.uniform())           # box half sizes
    px, py = -1.0 + 2.0 * rng.uniform(), -1.8 + 1.2 * rng.uniform()                     # robot below the box
    pth = 0.5 * math.pi + (-0.5 + rng.uniform())                                        # looking roughly "up"
    phi = -0.5 * math.pi + np.arange(R) * (math.pi / (R - 1))
    ang = pth[None, :] + phi[:, None]
    dx, dy = np.cos(ang), np.sin(ang)
    big = 1e9
    with np.errstate(divide="ignore", invalid="ignore"):
        # outer walls: the robot is inside, take the exit distance
        tx = np.where(dx > 0, (wx - px) / dx, np.where(dx < 0, (-wx - px) / dx, big))
        ty = np.where(dy > 0, (wy - py) / dy, np.where(dy < 0, (-wy - py) / dy, big))
        t_room = np.minimum(tx, ty)
        # box: slab test
        t1x, t2x = (bx - bw - px) / dx, (bx + bw - px) / dx
        t1y, t2y = (by - bh - py) / dy, (by + bh - py) / dy
        tnx, tfx = np.minimum(t1x, t2x), np.maximum(t1x, t2x)
        tny, tfy = np.minimum(t1y, t2y), np.maximum(t1y, t2y)
        tn, tf = np.maximum(tnx, tny), np.minimum(tfx, tfy)
        t_box = np.where((tn <= tf) & (tn > 0), tn, big)
    ranges = np.minimum(t_room, t_box)
    noise = np.stack([rng.normal() for _ in range(R)]) if range_sigma > 0 else 0.0
    ranges = ranges + range_sigma * noise

    # rasterise the map
    cc = (np.arange(G) + 0.5) * res - half                      # cell centres
    X, Y = np.meshgrid(cc, cc)                                  # [iy, ix]
    grid = np.zeros((N, G, G), dtype)
    for e in range(N):
        inside = (np.abs(X) < wx[e] - 0.25 * res) & (np.abs(Y) < wy[e] - 0.25 * res)
        wall = (np.abs(np.abs(X) - wx[e]) < 0.5 * res) & (np.abs(Y) <= wy[e] + 0.5 * res) | \
               (np.abs(np.abs(Y) - wy[e]) < 0.5 * res) & (np.abs(X) <= wx[e] + 0.5 * res)
        inbox = (np.abs(X - bx[e]) <= bw[e] + 0.5 * res) & (np.abs(Y - by[e]) <= bh[e] + 0.5 * res)
        boxwall = inbox & ~((np.abs(X - bx[e]) < bw[e] - 0.5 * res) & (np.abs(Y - by[e]) < bh[e] - 0.5 * res))
        g = np.where(inside, -l_lo, 0.0)
        g = np.where(inbox, 0.0, g)
        g = np.where(wall | boxwall, l_hi, g)
        grid[e] = g
    pose_true = np.stack([px, py, pth])
    ox, oy, ot = offset_cells
    pose_pred = np.stack([px - ox * res, py - oy * res, pth - ot * sth])
    return dict(grid=grid, ranges=ranges.astype(dtype), pose_true=pose_true.astype(dtype), pose_pred=pose_pred.astype(dtype),
                G=G, res=res, R=R)
