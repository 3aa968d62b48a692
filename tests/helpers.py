"""Shared test helpers: drive one oracle environment from generator arrays (float64 path)."""
import numpy as np


def step_inputs(data, t, env):
    """Inputs of step t (1-based) for one environment, as float64 numpy."""
    L = data["cfg"].L
    odom = data["odom"][t - 1, :, env].astype(np.float64)
    back = int(data["lc_back"][t - 1, env])
    zlc = data["lc_meas"][t - 1, :, env].astype(np.float64)
    valid, zrb = rb_inputs(data, t, env)
    return odom, back, zlc, valid, zrb


def rb_inputs(data, t, env):
    L = data["cfg"].L
    if L == 0:
        return None, None
    valid = np.array([(int(data["rb_mask"][t, l // 32, env]) >> (l % 32)) & 1 for l in range(L)], np.int32)
    zrb = data["rb_meas"][t, :, :, env].astype(np.float64).T.copy()  # [L][2]
    return valid, zrb


def drive(orc, data, env, iters, on_step=None, steps=None):
    """reset -> (observe_first) -> for t: push, solve, cov, [marginalize iff full] (R19)."""
    W = data["cfg"].W
    T = data["T"] if steps is None else steps
    orc.reset()
    if data["cfg"].L:
        orc.observe_first(*rb_inputs(data, 0, env))
    out = []
    for t in range(1, T + 1):
        odom, back, zlc, valid, zrb = step_inputs(data, t, env)
        if data.get("reset") is not None and data["reset"][t - 1, env]:
            orc.reset(data["reset_pose"][t - 1, :, env].astype(np.float64))
        orc.push(odom, back, zlc, valid, zrb)
        un = unary_inputs(data, t, env)
        if un is not None:
            orc.add_unary(*un)
        sn = orc.solve(iters)
        S, ld = orc.cov()
        P = orc.poses()
        rec = dict(t=t, step=sn, cov=S, logdet=ld, poses=P, count=orc.count)
        if on_step is not None:
            on_step(rec, orc)
        out.append(rec)
        if orc.count == W:
            orc.marginalize()
    return out


def unary_inputs(data, t, env):
    """(pose3, info3x3) of the unary factor of step t, or None."""
    if data.get("un_valid") is None or not data["un_valid"][t - 1, env]:
        return None
    z = data["un_pose"][t - 1, :, env].astype(np.float64)
    i6 = data["un_info"][t - 1, :, env].astype(np.float64)
    Om = np.array([[i6[0], i6[1], i6[3]], [i6[1], i6[2], i6[4]], [i6[3], i6[4], i6[5]]])
    return z, Om
