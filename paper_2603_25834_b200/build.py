"""Builds the C-ABI CUDA library ``libslam_b200.so`` in-tree with nvcc for sm_100a: one object per source file
(rebuilt only when that file or a header changed), then one link."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libslam_b200.so")
SOURCES = ["slam_api.cu", "slam_scan.cu"]
HEADERS = ["slam_kernels.cuh", "slam_ref64.cuh", "slam_layout.h", os.path.join("..", "..", "include", "slam.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _stale(target: str, src: str) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return os.path.getmtime(src) > t or _newest_header() > t


def needs_build() -> bool:
    return any(_stale(LIB, os.path.join(CSRC, s)) for s in SOURCES)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    objs, procs = [], []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, src):
            cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, cmd)
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", LIB])
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
