"""Drives the CUDA library over a generated workload (used by the GPU parity tests and smoke())."""
import numpy as np
import torch

from harness import synth  # noqa: F401  (kept for callers)


def to_dev(data, device="cuda:0"):
    """Uploads the step inputs of a synth.generate() dict; returns a dict of device tensors."""
    d = {}
    d["odom"] = torch.from_numpy(np.ascontiguousarray(data["odom"], dtype=np.float32)).to(device)
    d["lc_back"] = torch.from_numpy(np.ascontiguousarray(data["lc_back"], dtype=np.int32)).to(device)
    d["lc_meas"] = torch.from_numpy(np.ascontiguousarray(data["lc_meas"], dtype=np.float32)).to(device)
    d["rb_mask"] = torch.from_numpy(np.ascontiguousarray(data["rb_mask"]).view(np.int32)).to(device)
    d["rb_meas"] = torch.from_numpy(np.ascontiguousarray(data["rb_meas"], dtype=np.float32)).to(device)
    if data.get("un_valid") is not None:
        d["un_valid"] = torch.from_numpy(np.ascontiguousarray(data["un_valid"], dtype=np.int32)).to(device)
        d["un_pose"] = torch.from_numpy(np.ascontiguousarray(data["un_pose"], dtype=np.float32)).to(device)
        d["un_info"] = torch.from_numpy(np.ascontiguousarray(data["un_info"], dtype=np.float32)).to(device)
    if data.get("reset") is not None:
        d["reset"] = torch.from_numpy(np.ascontiguousarray(data["reset"], dtype=np.int32)).to(device)
        d["reset_pose"] = torch.from_numpy(np.ascontiguousarray(data["reset_pose"], dtype=np.float32)).to(device)
    return d


def run_gpu(slam, data, iters, fused=True, steps=None, want_poses=True):
    """reset -> (observe_first) -> T x [push, solve, cov, dopt, (marginalize iff full)] through the C ABI.

    Returns numpy arrays poses[T,N,W,3] (global), cov[T,N,3,3], logdet[T,N], status[N]; the fused path
    (one slam_step per step) returns last_pose[T,N,3] (newest pose, global) instead of the whole window."""
    cfg = data["cfg"]
    T = data["T"] if steps is None else steps
    N, W, L = slam.N, slam.W, slam.L
    dev = to_dev(data, slam.device)
    slam.reset()
    if L:
        slam.observe_first(dev["rb_mask"][0], dev["rb_meas"][0])
    cov = torch.zeros(T, 9, N, device=slam.device)
    logdet = torch.zeros(T, N, device=slam.device)
    poses = torch.zeros(T, 3, W, N, device=slam.device) if want_poses else None
    last = torch.zeros(T, 3, N, device=slam.device) if (fused and not want_poses) else None
    for t in range(1, T + 1):
        args = (dev["odom"][t - 1], dev["lc_back"][t - 1], dev["lc_meas"][t - 1],
                dev["rb_mask"][t] if L else None, dev["rb_meas"][t] if L else None)
        if "reset" in dev:
            slam.reset_envs(dev["reset"][t - 1], dev["reset_pose"][t - 1])
        if "un_valid" in dev:
            slam.set_unary(dev["un_pose"][t - 1], dev["un_info"][t - 1], dev["un_valid"][t - 1])
        if fused and not want_poses:
            slam.step(*args, iters=iters, cov=cov[t - 1], logdet=logdet[t - 1], last_pose=last[t - 1])
        else:
            slam.push_step(*args)
            slam.solve(iters)
            slam.marginal_cov(cov[t - 1])
            slam.dopt(logdet[t - 1])
            if want_poses:
                slam.get_poses(poses[t - 1])
            if slam.count == W:
                slam.marginalize_oldest()
    torch.cuda.synchronize()
    out = dict(cov=cov.cpu().numpy().reshape(T, 3, 3, N).transpose(0, 3, 1, 2).astype(np.float64),
               logdet=logdet.cpu().numpy().astype(np.float64), status=slam.get_status().cpu().numpy())
    if want_poses:
        out["poses"] = poses.cpu().numpy().transpose(0, 3, 2, 1).astype(np.float64)
    if last is not None:
        out["last_pose"] = last.cpu().numpy().transpose(0, 2, 1).astype(np.float64)
    return out


def wrap(x):
    return np.arctan2(np.sin(x), np.cos(x))


def parity_errors(gpu, ref, counts=None):
    """Normalised errors per (step, env) in units of the tolerances of DESIGN.md R23 (1.0 = at tolerance):
    poses: max_k |dx_k|_inf / (1e-4 max(1, max_k |x_k|_inf)), angles wrapped;
    cov:   max_ij |dS_ij| / (1e-3 sqrt(S_ii S_jj)) with the oracle's S;  logdet: |d| / 1e-3."""
    out = {}
    if gpu.get("last_pose") is not None and ref.get("poses") is not None:
        # newest pose of the window after the solve of step t: slot min(t + 1, W) - 1 (or `counts` - 1 per env)
        T, ne, W, _ = ref["poses"].shape
        c = np.minimum(np.arange(T) + 2, W)[:, None] * np.ones((1, ne), int) if counts is None else counts
        newest = np.take_along_axis(ref["poses"], (c - 1)[:, :, None, None].repeat(3, axis=3), axis=2)[:, :, 0]
        d = gpu["last_pose"] - newest
        d[..., 2] = wrap(d[..., 2])
        scale = np.maximum(1.0, np.abs(ref["poses"]).max(axis=(2, 3)))
        out["last_pose"] = np.abs(d).max(axis=2) / (1e-4 * scale)
    if "poses" in gpu and gpu["poses"] is not None and ref.get("poses") is not None:
        d = gpu["poses"] - ref["poses"]
        d[..., 2] = wrap(d[..., 2])
        scale = np.maximum(1.0, np.abs(ref["poses"]).max(axis=(2, 3)))
        out["poses"] = np.abs(d).max(axis=(2, 3)) / (1e-4 * scale)
    S = ref["cov"]
    dg = np.sqrt(np.einsum("tnii->tni", S))
    sc = dg[..., :, None] * dg[..., None, :]
    out["cov"] = (np.abs(gpu["cov"] - S) / (1e-3 * sc)).max(axis=(2, 3))
    out["logdet"] = np.abs(gpu["logdet"] - ref["logdet"]) / 1e-3
    return out
