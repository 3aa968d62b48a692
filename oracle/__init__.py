"""ctypes wrapper of the fp64 CPU oracle (``slam_oracle.c``) -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It never imports the CUDA product package (and vice versa).
``build()`` compiles the C source with gcc (``-O2 -fopenmp``); building the checker is not using it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "slam_oracle.c")
_HDR = os.path.join(_HERE, "slam_oracle.h")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

DEFAULT_SIGMAS = (0.01, 0.01, 0.005, 0.05, 0.05, 0.02, 0.10, 0.10, 0.03, 0.05, 0.01)

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, _dp, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_reset.argtypes = [C.c_void_p, _dp]
        L.orc_count.argtypes = [C.c_void_p]
        L.orc_dim.argtypes = [C.c_void_p]
        L.orc_push.argtypes = [C.c_void_p, _dp, C.c_int, _dp, _ip, _dp]
        L.orc_observe_first.argtypes = [C.c_void_p, _ip, _dp]
        L.orc_solve.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc_cov.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_marginalize.argtypes = [C.c_void_p]
        L.orc_get_poses.argtypes = [C.c_void_p, _dp]
        L.orc_get_landmarks.argtypes = [C.c_void_p, _dp, _ip]
        L.orc_get_state.argtypes = [C.c_void_p, _dp]
        L.orc_set_state.argtypes = [C.c_void_p, _dp]
        L.orc_get_prior.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_assemble.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_cost.restype = C.c_double
        L.orc_cost.argtypes = [C.c_void_p]
        L.orc_between_factor.argtypes = [_dp, _dp, _dp, C.c_int, _dp, _dp, _dp]
        L.orc_rb_factor.argtypes = [_dp, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_reanchor_map.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_reanchor_jac.argtypes = [C.c_void_p, _dp]
        L.orc_add_unary.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_unary_factor.argtypes = [_dp, _dp, _dp, C.c_int, _dp, _dp, _dp]
        L.orc_batch_set_unary.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_batch_set_unary.restype = None
        L.orc_batch_set_resets.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_batch_set_resets.restype = None
        L.orc_run_batch.restype = C.c_int
        L.orc_run_batch.argtypes = [C.c_int] * 5 + [_dp, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                                    C.c_void_p, _ip, C.c_int, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    """One environment of the fp64 oracle."""

    def __init__(self, W: int, L: int = 0, sigmas=DEFAULT_SIGMAS, linear: bool = False):
        self.W, self.L, self.n = W, L, 3 * W + 2 * L
        self._sig = _d(sigmas)
        self._h = lib().orc_create(W, L, _p(self._sig), int(linear))
        if not self._h:
            raise ValueError("orc_create failed")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    @property
    def count(self) -> int:
        return lib().orc_count(self._h)

    def reset(self, init_pose=None):
        ip = None if init_pose is None else _d(init_pose)
        lib().orc_reset(self._h, None if ip is None else _p(ip))

    def _rb(self, rb_valid, rb_meas):
        if self.L == 0 or rb_valid is None:
            return None, None, None, None
        v = np.ascontiguousarray(rb_valid, dtype=np.int32)
        z = _d(rb_meas).reshape(self.L, 2)
        return v, z, v.ctypes.data_as(_ip), _p(z)

    def push(self, odom, lc_back=0, lc_meas=None, rb_valid=None, rb_meas=None):
        od = _d(odom)
        zl = _d(lc_meas if lc_meas is not None else (0, 0, 0))
        v, z, vp, zp = self._rb(rb_valid, rb_meas)
        rc = lib().orc_push(self._h, _p(od), int(lc_back), _p(zl), vp, zp)
        if rc != 0:
            raise RuntimeError("push on a full window")

    def observe_first(self, rb_valid, rb_meas):
        v, z, vp, zp = self._rb(rb_valid, rb_meas)
        if lib().orc_observe_first(self._h, vp, zp) != 0:
            raise RuntimeError("observe_first after a push")

    def add_unary(self, pose, info):
        """Unary absolute-pose factor on the newest pose: measured global pose (3), 3x3 information."""
        z, om = _d(pose), _d(np.asarray(info, float).reshape(3, 3))
        lib().orc_add_unary(self._h, _p(z), _p(om))

    def solve(self, iters: int) -> float:
        s = C.c_double(0.0)
        if lib().orc_solve(self._h, iters, C.byref(s)) != 0:
            raise np.linalg.LinAlgError("singular H")
        return s.value

    def cov(self):
        S = np.zeros(9)
        ld = C.c_double(0.0)
        if lib().orc_cov(self._h, _p(S), C.byref(ld)) != 0:
            raise np.linalg.LinAlgError("singular H")
        return S.reshape(3, 3), ld.value

    def marginalize(self):
        rc = lib().orc_marginalize(self._h)
        if rc != 0:
            raise RuntimeError("marginalize failed")

    def poses(self):
        P = np.zeros((self.W, 3))
        lib().orc_get_poses(self._h, _p(P))
        return P

    def landmarks(self):
        lm = np.zeros((max(self.L, 1), 2))
        act = np.zeros(max(self.L, 1), np.int32)
        lib().orc_get_landmarks(self._h, _p(lm), act.ctypes.data_as(_ip))
        return lm[: self.L], act[: self.L]

    def state(self):
        v = np.zeros(self.n)
        lib().orc_get_state(self._h, _p(v))
        return v

    def set_state(self, v):
        v = _d(v)
        lib().orc_set_state(self._h, _p(v))

    def prior(self):
        Lam, g, vb = np.zeros((self.n, self.n)), np.zeros(self.n), np.zeros(self.n)
        lib().orc_get_prior(self._h, _p(Lam), _p(g), _p(vb))
        return Lam, g, vb

    def assemble(self):
        H, b = np.zeros((self.n, self.n)), np.zeros(self.n)
        lib().orc_assemble(self._h, _p(H), _p(b))
        return H, b

    def cost(self) -> float:
        return lib().orc_cost(self._h)

    def reanchor_map(self, v):
        v = _d(v)
        u = np.zeros(self.n)
        lib().orc_reanchor_map(self._h, _p(v), _p(u))
        return u

    def reanchor_jac(self):
        M = np.zeros((self.n, self.n))
        lib().orc_reanchor_jac(self._h, _p(M))
        return M


def between_factor(ei, ej, z, i_is_frame=False):
    r, Ji, Jj = np.zeros(3), np.zeros(9), np.zeros(9)
    lib().orc_between_factor(_p(_d(ei)), _p(_d(ej)), _p(_d(z)), int(i_is_frame), _p(r), _p(Ji), _p(Jj))
    return r, Ji.reshape(3, 3), Jj.reshape(3, 3)


def rb_factor(a, ek, gl, z, k_is_frame=False):
    """Range-bearing factor, landmark gl global, observing pose a (+) ek: returns r, Ja (2x3), Jp (2x3), Jg (2x2)."""
    r, Ja, Jp, Jg = np.zeros(2), np.zeros(6), np.zeros(6), np.zeros(4)
    lib().orc_rb_factor(_p(_d(a)), _p(_d(ek)), _p(_d(gl)), _p(_d(z)), int(k_is_frame), _p(r), _p(Ja), _p(Jp), _p(Jg))
    return r, Ja.reshape(2, 3), Jp.reshape(2, 3), Jg.reshape(2, 2)


def unary_factor(a, ek, z, k_is_frame=False):
    r, Ja, Je = np.zeros(3), np.zeros(9), np.zeros(9)
    lib().orc_unary_factor(_p(_d(a)), _p(_d(ek)), _p(_d(z)), int(k_is_frame), _p(r), _p(Ja), _p(Je))
    return r, Ja.reshape(3, 3), Je.reshape(3, 3)


def max_threads() -> int:
    return lib().orc_max_threads()


def run_batch(data: dict, iters: int, envs=None, sigmas=DEFAULT_SIGMAS, threads: int = 0,
              want=("poses", "cov", "logdet", "step"), f32_storage: bool = False) -> dict:
    """Run push -> solve -> cov -> (marginalize iff full) over ``data`` (a ``synth.generate`` dict, float32
    arrays) for the environments ``envs`` (column indices into the arrays).  Returns float64 arrays
    ``poses[T,ne,W,3]``, ``cov[T,ne,3,3]``, ``logdet[T,ne]``, ``step[T,ne]`` and ``bad`` (#singular envs)."""
    cfg = data["cfg"]
    W, L, T = cfg.W, cfg.L, data["T"]
    N = data["odom"].shape[-1]
    envs = np.arange(N, dtype=np.int32) if envs is None else np.ascontiguousarray(envs, dtype=np.int32)
    ne = len(envs)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    odom, lc_meas, rb_meas = f32(data["odom"]), f32(data["lc_meas"]), f32(data["rb_meas"])
    lc_back = np.ascontiguousarray(data["lc_back"], dtype=np.int32)
    rb_mask = np.ascontiguousarray(data["rb_mask"], dtype=np.uint32)
    out = {}
    out["poses"] = np.zeros((T, ne, W, 3)) if "poses" in want else None
    out["cov"] = np.zeros((T, ne, 3, 3)) if "cov" in want else None
    out["logdet"] = np.zeros((T, ne)) if "logdet" in want else None
    out["step"] = np.zeros((T, ne)) if "step" in want else None
    sig = _d(sigmas)
    ptr = lambda a: None if a is None else _p(a)
    vp = lambda a: a.ctypes.data_as(C.c_void_p)
    keep = None
    if data.get("un_valid") is not None:
        keep = (np.ascontiguousarray(data["un_valid"], dtype=np.int32), f32(data["un_pose"]), f32(data["un_info"]))
        lib().orc_batch_set_unary(vp(keep[0]), vp(keep[1]), vp(keep[2]))
    keep2 = None
    if data.get("reset") is not None:
        keep2 = (np.ascontiguousarray(data["reset"], dtype=np.int32), f32(data["reset_pose"]))
        lib().orc_batch_set_resets(vp(keep2[0]), vp(keep2[1]))
    lib().orc_batch_set_f32_storage(int(f32_storage))
    bad = lib().orc_run_batch(N, W, L, T, iters, _p(sig), vp(odom), vp(lc_back), vp(lc_meas), vp(rb_mask),
                              vp(rb_meas), envs.ctypes.data_as(_ip), ne, int(threads),
                              ptr(out["poses"]), ptr(out["cov"]), ptr(out["logdet"]), ptr(out["step"]))
    lib().orc_batch_set_f32_storage(0)
    lib().orc_batch_set_unary(None, None, None)
    lib().orc_batch_set_resets(None, None)
    out["bad"] = bad
    return out
