"""Thin Python binding of the C-ABI library (``include/slam.h``): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``csrc/``; PyTorch is used for device memory
and streams.  There is NO CPU fallback: if ``libslam_b200.so`` is missing and cannot be built with
nvcc, importing this module raises.  Method names follow the C entry points.
"""
from __future__ import annotations

import ctypes as C
import os
import shutil

import torch

from . import build as _build

SLAM_OK, SLAM_EINVAL, SLAM_ESTATE, SLAM_ENOMEM, SLAM_ECUDA = 0, 1, 2, 3, 4
SLAM_ENV_NOT_PD, SLAM_ENV_NONFINITE, SLAM_ENV_INTERNAL = 1, 2, 4
_ERR = {1: "SLAM_EINVAL", 2: "SLAM_ESTATE", 3: "SLAM_ENOMEM", 4: "SLAM_ECUDA"}

# every symbol include/slam.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "slam_default_config", "slam_workspace_bytes", "slam_create", "slam_destroy", "slam_reset",
    "slam_reset_envs", "slam_push_step", "slam_set_unary", "slam_observe_first", "slam_solve", "slam_marginal_cov", "slam_dopt",
    "slam_marginalize_oldest", "slam_step", "slam_step_host", "slam_get_poses", "slam_get_landmarks",
    "slam_get_status", "slam_get_stats", "slam_set_precision", "slam_run_static", "slam_fma_probe", "slam_kernel_timing", "slam_kernel_timing_read", "slam_reward", "slam_scan_match", "slam_grid_update", "slam_count", "slam_launch_count", "slam_last_error", "slam_kernel_info",
)


class SlamConfig(C.Structure):
    _fields_ = [("prior_sigma", C.c_float * 3), ("odo_sigma", C.c_float * 3), ("lc_sigma", C.c_float * 3),
                ("rb_sigma", C.c_float * 2)]


class RewardParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("lambda_col", "lambda_explore", "lambda_abs", "lambda_delta", "u_hi", "kappa",
                                         "d_crash", "d_full")]


class ScanParams(C.Structure):
    _fields_ = [("G", C.c_int), ("res", C.c_float), ("R", C.c_int), ("r_min", C.c_float), ("r_max", C.c_float),
                ("hx", C.c_int), ("hy", C.c_int), ("ht", C.c_int), ("sxy", C.c_float), ("sth", C.c_float)]


class SlamError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERR.get(code, code)}: {msg}")
        self.code = code


def _load() -> C.CDLL:
    path = _build.LIB
    if _build.needs_build():
        if shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc"):
            _build.build()
        elif not os.path.exists(path):
            raise ImportError(f"{path} is missing and nvcc is not available: build it with __graft_entry__.build()")
    lib = C.CDLL(path)
    vp, fp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    lib.slam_default_config.argtypes = [C.POINTER(SlamConfig)]
    lib.slam_default_config.restype = None
    lib.slam_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int]
    lib.slam_workspace_bytes.restype = C.c_size_t
    lib.slam_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.POINTER(SlamConfig), vp, C.c_size_t, vp]
    lib.slam_destroy.argtypes = [vp]
    lib.slam_destroy.restype = None
    lib.slam_reset.argtypes = [vp, fp]
    lib.slam_reset_envs.argtypes = [vp, ip, fp]
    lib.slam_push_step.argtypes = [vp, fp, ip, fp, ip, fp]
    lib.slam_set_unary.argtypes = [vp, fp, fp, ip]
    lib.slam_observe_first.argtypes = [vp, ip, fp]
    lib.slam_solve.argtypes = [vp, C.c_int]
    lib.slam_marginal_cov.argtypes = [vp, fp]
    lib.slam_dopt.argtypes = [vp, fp, fp]
    lib.slam_marginalize_oldest.argtypes = [vp]
    lib.slam_step.argtypes = [vp, fp, ip, fp, ip, fp, C.c_int, fp, fp, fp]
    lib.slam_step_host.argtypes = [vp, fp, ip, fp, ip, fp, C.c_int, fp, fp, fp]
    lib.slam_get_poses.argtypes = [vp, fp]
    lib.slam_get_landmarks.argtypes = [vp, fp, ip]
    lib.slam_get_status.argtypes = [vp, ip]
    lib.slam_get_stats.argtypes = [vp, ip]
    lib.slam_reward.argtypes = [vp, C.POINTER(RewardParams), fp, fp, fp, fp, ip, fp]
    lib.slam_scan_match.argtypes = [C.POINTER(ScanParams), C.c_int, fp, fp, fp, fp, fp, fp, vp]
    lib.slam_grid_update.argtypes = [C.POINTER(ScanParams), C.c_int, fp, fp, fp, fp, C.c_float, C.c_float, C.c_float, vp]
    lib.slam_set_precision.argtypes = [vp, C.c_int, C.c_float, C.c_float]
    lib.slam_run_static.argtypes = [C.c_int] * 5 + [C.POINTER(SlamConfig), fp, ip, fp, ip, fp, fp, fp, fp, vp, C.c_char_p, C.c_size_t]
    lib.slam_kernel_timing.argtypes = [vp, C.c_int]
    lib.slam_kernel_timing_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    lib.slam_fma_probe.argtypes = [C.c_longlong, fp, vp, C.POINTER(C.c_double)]
    lib.slam_count.argtypes = [vp]
    lib.slam_launch_count.argtypes = [vp]
    lib.slam_launch_count.restype = C.c_longlong
    lib.slam_last_error.argtypes = [vp]
    lib.slam_last_error.restype = C.c_char_p
    lib.slam_kernel_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    return lib


LIB = _load()


def default_config() -> SlamConfig:
    cfg = SlamConfig()
    LIB.slam_default_config(C.byref(cfg))
    return cfg


def workspace_bytes(batch: int, window: int, landmarks: int) -> int:
    return int(LIB.slam_workspace_bytes(batch, window, landmarks))


def _f32(t, shape, name):
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise SlamError(SLAM_EINVAL, f"{name}: expected contiguous float32 CUDA tensor of shape {tuple(shape)}")
    return C.c_void_p(t.data_ptr())


def scan_match(par: ScanParams, grid, pose_pred, ranges):
    """NEXT-3: returns (pose_meas [3,N], score [N], second [N])."""
    N = grid.shape[0]
    meas = torch.empty(3, N, device=grid.device)
    s1 = torch.empty(N, device=grid.device)
    s2 = torch.empty(N, device=grid.device)
    rc = LIB.slam_scan_match(C.byref(par), N, _f32(grid, (N, par.G, par.G), "grid"), _f32(pose_pred, (3, N), "pose_pred"),
                             _f32(ranges, (par.R, N), "ranges"), C.c_void_p(meas.data_ptr()), C.c_void_p(s1.data_ptr()),
                             C.c_void_p(s2.data_ptr()), C.c_void_p(torch.cuda.current_stream(grid.device).cuda_stream))
    if rc != SLAM_OK:
        raise SlamError(rc, "slam_scan_match")
    return meas, s1, s2


def grid_update(par: ScanParams, grid, pose, ranges, weight, l_free: float, l_occ: float, l_clamp: float):
    """NEXT-3: in-place confidence-weighted log-odds update of `grid`."""
    N = grid.shape[0]
    rc = LIB.slam_grid_update(C.byref(par), N, _f32(grid, (N, par.G, par.G), "grid"), _f32(pose, (3, N), "pose"),
                              _f32(ranges, (par.R, N), "ranges"), _f32(weight, (N,), "weight"), l_free, l_occ, l_clamp,
                              C.c_void_p(torch.cuda.current_stream(grid.device).cuda_stream))
    if rc != SLAM_OK:
        raise SlamError(rc, "slam_grid_update")
    return grid


def fma_probe(iters: int, device="cuda:0") -> float:
    """slam_fma_probe: enqueues one launch of the register-resident FP32 FMA kernel on `device`'s current stream and
    returns the floating-point operations that launch performs (the caller times it with CUDA events)."""
    dev = torch.device(device)
    sink = torch.zeros(1, device=dev)
    flops = C.c_double(0.0)
    with torch.cuda.device(dev):
        rc = LIB.slam_fma_probe(int(iters), C.c_void_p(sink.data_ptr()), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                C.byref(flops))
    if rc != SLAM_OK:
        raise SlamError(rc, "slam_fma_probe")
    return float(flops.value)


STATIC_MAX_BYTES = 16 << 20


def run_static(batch: int, window: int, landmarks: int, iters: int, odom, lc_back=None, lc_meas=None, rb_mask=None,
               rb_meas=None, cov=None, logdet=None, last_pose=None, config: SlamConfig | None = None):
    """slam_run_static: one whole episode on the library's static scratch array (no device allocation in the library;
    inputs and outputs are the caller's tensors: odom [T,3,N], lc_back [T,N], lc_meas [T,3,N], rb_mask [T+1,nw,N],
    rb_meas [T+1,2,L,N], cov [T,9,N], logdet [T,N], last_pose [T,3,N])."""
    T, dev = int(odom.shape[0]), odom.device
    ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())
    for t in (odom, lc_back, lc_meas, rb_mask, rb_meas, cov, logdet, last_pose):
        if t is not None and (not t.is_cuda or t.device != dev or not t.is_contiguous()):
            raise SlamError(SLAM_EINVAL, "run_static: contiguous CUDA tensors on one device expected")
    msg = C.create_string_buffer(256)
    with torch.cuda.device(dev):
        rc = LIB.slam_run_static(int(batch), int(window), int(landmarks), T, int(iters),
                                 C.byref(config) if config is not None else None, ptr(odom), ptr(lc_back), ptr(lc_meas),
                                 ptr(rb_mask), ptr(rb_meas), ptr(cov), ptr(logdet), ptr(last_pose),
                                 C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), msg, 256)
    if rc != SLAM_OK:
        raise SlamError(rc, msg.value.decode())


class FixedLagSlam:
    """One context = `batch` environments in lock-step on one CUDA stream."""

    def __init__(self, batch: int, window: int, landmarks: int = 0, config: SlamConfig | None = None,
                 device: str | torch.device = "cuda:0", stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("FixedLagSlam needs a CUDA device (there is no CPU fallback)")
        self.N, self.W, self.L = int(batch), int(window), int(landmarks)
        self.nw = (self.L + 31) // 32
        self.device = torch.device(device)
        nbytes = workspace_bytes(self.N, self.W, self.L)
        if nbytes == 0:
            raise SlamError(SLAM_EINVAL, f"invalid sizes batch={batch} window={window} landmarks={landmarks}")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            h = C.c_void_p()
            rc = LIB.slam_create(C.byref(h), self.N, self.W, self.L, C.byref(config) if config is not None else None,
                                 C.c_void_p(self._ws_ptr), nbytes, C.c_void_p(self.stream.cuda_stream))
        if rc != SLAM_OK:
            raise SlamError(rc, "slam_create failed")
        self._h = h

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            LIB.slam_destroy(h)
            self._h = None

    # ---- marshalling helpers
    def _chk(self, rc: int):
        if rc != SLAM_OK:
            raise SlamError(rc, (LIB.slam_last_error(self._h) or b"").decode())

    def _dev(self, t, shape, dtypes, name):
        if t is None:
            return None
        if not isinstance(t, torch.Tensor) or t.device != self.device or t.dtype not in dtypes or not t.is_contiguous() \
                or tuple(t.shape) != tuple(shape):
            raise SlamError(SLAM_EINVAL, f"{name}: expected contiguous {dtypes[0]} tensor of shape {tuple(shape)} on {self.device}")
        return C.c_void_p(t.data_ptr())

    def _host(self, t, shape, dtypes, name):
        if t is None:
            return None
        if not isinstance(t, torch.Tensor) or t.device.type != "cpu" or t.dtype not in dtypes or not t.is_contiguous() \
                or tuple(t.shape) != tuple(shape):
            raise SlamError(SLAM_EINVAL, f"{name}: expected contiguous host {dtypes[0]} tensor of shape {tuple(shape)}")
        return C.c_void_p(t.data_ptr())

    def _new(self, *shape, dtype=torch.float32):
        return torch.empty(shape, dtype=dtype, device=self.device)

    _F = (torch.float32,)
    _I = (torch.int32,)
    _U = (torch.int32, torch.uint32)

    def _push_ptrs(self, conv, odom, lc_back, lc_meas, rb_mask, rb_meas):
        N, L = self.N, self.L
        return (conv(odom, (3, N), self._F, "odom"), conv(lc_back, (N,), self._I, "lc_back"),
                conv(lc_meas, (3, N), self._F, "lc_meas"),
                conv(rb_mask, (self.nw, N), self._U, "rb_mask") if L else None,
                conv(rb_meas, (2, L, N), self._F, "rb_meas") if L else None)

    # ---- the C entry points
    def reset(self, init_pose=None):
        self._chk(LIB.slam_reset(self._h, self._dev(init_pose, (3, self.N), self._F, "init_pose")))

    def reset_envs(self, mask, init_pose=None):
        self._chk(LIB.slam_reset_envs(self._h, self._dev(mask, (self.N,), self._I, "mask"),
                                      self._dev(init_pose, (3, self.N), self._F, "init_pose")))

    def push_step(self, odom, lc_back=None, lc_meas=None, rb_mask=None, rb_meas=None):
        self._chk(LIB.slam_push_step(self._h, *self._push_ptrs(self._dev, odom, lc_back, lc_meas, rb_mask, rb_meas)))

    def set_unary(self, pose, info, valid=None):
        """Unary absolute-pose factor for the pose appended by the next push_step / step (keep the tensors alive)."""
        self._unary_keep = (pose, info, valid)
        self._chk(LIB.slam_set_unary(self._h, self._dev(pose, (3, self.N), self._F, "pose"),
                                     self._dev(info, (6, self.N), self._F, "info"),
                                     self._dev(valid, (self.N,), self._I, "valid")))

    def observe_first(self, rb_mask, rb_meas):
        if self.L == 0:
            return
        self._chk(LIB.slam_observe_first(self._h, self._dev(rb_mask, (self.nw, self.N), self._U, "rb_mask"),
                                         self._dev(rb_meas, (2, self.L, self.N), self._F, "rb_meas")))

    def solve(self, iters: int):
        self._chk(LIB.slam_solve(self._h, int(iters)))

    def marginal_cov(self, out=None):
        out = self._new(9, self.N) if out is None else out
        self._chk(LIB.slam_marginal_cov(self._h, self._dev(out, (9, self.N), self._F, "cov")))
        return out

    def dopt(self, logdet=None, dopt=None):
        logdet = self._new(self.N) if logdet is None else logdet
        dopt = self._new(self.N) if dopt is None else dopt
        self._chk(LIB.slam_dopt(self._h, self._dev(logdet, (self.N,), self._F, "logdet"),
                                self._dev(dopt, (self.N,), self._F, "dopt")))
        return logdet, dopt

    def marginalize_oldest(self):
        self._chk(LIB.slam_marginalize_oldest(self._h))

    def step(self, odom, lc_back=None, lc_meas=None, rb_mask=None, rb_meas=None, *, iters: int, cov=None, logdet=None,
             last_pose=None):
        ptrs = self._push_ptrs(self._dev, odom, lc_back, lc_meas, rb_mask, rb_meas)
        self._chk(LIB.slam_step(self._h, *ptrs, int(iters), self._dev(cov, (9, self.N), self._F, "cov"),
                                self._dev(logdet, (self.N,), self._F, "logdet"),
                                self._dev(last_pose, (3, self.N), self._F, "last_pose")))

    def step_host(self, odom, lc_back=None, lc_meas=None, rb_mask=None, rb_meas=None, *, iters: int, cov=None,
                  logdet=None, last_pose=None):
        ptrs = self._push_ptrs(self._host, odom, lc_back, lc_meas, rb_mask, rb_meas)
        self._chk(LIB.slam_step_host(self._h, *ptrs, int(iters), self._host(cov, (9, self.N), self._F, "cov"),
                                     self._host(logdet, (self.N,), self._F, "logdet"),
                                     self._host(last_pose, (3, self.N), self._F, "last_pose")))

    def get_poses(self, out=None):
        out = self._new(3, self.W, self.N) if out is None else out
        self._chk(LIB.slam_get_poses(self._h, self._dev(out, (3, self.W, self.N), self._F, "poses")))
        return out

    def get_landmarks(self):
        lm = self._new(2, max(self.L, 1), self.N)[:, : self.L].contiguous()
        act = self._new(max(self.nw, 1), self.N, dtype=torch.int32)[: self.nw].contiguous()
        if self.L:
            self._chk(LIB.slam_get_landmarks(self._h, C.c_void_p(lm.data_ptr()), C.c_void_p(act.data_ptr())))
        return lm, act

    def get_status(self):
        out = self._new(self.N, dtype=torch.int32)
        self._chk(LIB.slam_get_status(self._h, C.c_void_p(out.data_ptr())))
        return out

    def get_stats(self) -> dict:
        out = self._new(8, dtype=torch.int64)
        self._chk(LIB.slam_get_stats(self._h, C.c_void_p(out.data_ptr())))
        v = [int(x) for x in out.cpu()]
        return dict(max_envelope_words=v[0], mean_envelope_words=v[1] / max(v[2], 1), solved=v[2], waited=v[3], fp64_calls=v[4])

    def set_precision(self, mode: int, ratio_hi: float = 0.0, ratio_lo: float = 0.0):
        """-1 default rule, 0 fp32 only, 1 fp32 + fp64 fallback on ill-conditioned windows, 2 fp64 everywhere."""
        self._chk(LIB.slam_set_precision(self._h, int(mode), float(ratio_hi), float(ratio_lo)))

    def kernel_timing(self, max_steps: int):
        """Record per-kernel events for the next `max_steps` step launches (0: off)."""
        self._chk(LIB.slam_kernel_timing(self._h, int(max_steps)))

    def kernel_timing_read(self) -> dict:
        """Summed device milliseconds per kernel of the recorded step launches (synchronises)."""
        ms, n = (C.c_double * 3)(), C.c_int()
        self._chk(LIB.slam_kernel_timing_read(self._h, ms, C.byref(n)))
        return dict(step_kernel_ms=ms[0], ref64_kernel_ms=ms[1], order_kernel_ms=ms[2], steps=n.value)

    def reward(self, params: RewardParams, u, u_prev, dcells, d_min, collision, out=None):
        out = self._new(self.N) if out is None else out
        d = lambda x, n, ty=None: self._dev(x, (self.N,), ty or self._F, n)
        self._chk(LIB.slam_reward(self._h, C.byref(params), d(u, "u"), d(u_prev, "u_prev"), d(dcells, "dcells"),
                                  d(d_min, "d_min"), d(collision, "collision", self._I), d(out, "reward")))
        return out

    @property
    def count(self) -> int:
        return int(LIB.slam_count(self._h))

    @property
    def launch_count(self) -> int:
        return int(LIB.slam_launch_count(self._h))

    def kernel_info(self) -> dict:
        a, b, c = C.c_int(), C.c_int(), C.c_int()
        self._chk(LIB.slam_kernel_info(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return dict(smem_bytes_per_cta=a.value, warps_per_cta=b.value, ctas_per_sm=c.value)
