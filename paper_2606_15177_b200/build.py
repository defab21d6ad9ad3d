"""Build libgimbal.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

The translation units under csrc/ are compiled in parallel (one per expert count for the
router GEMM / gating kernels) and linked into one shared library with a static CUDA runtime.
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libgimbal.so")
SOURCES = ["gimbal_api.cu", "host_common.cu", "route_e16.cu", "route_e32.cu", "route_e64.cu", "route_e128.cu",
           "route_e256.cu"]
HEADERS = ["ptx.cuh", "gating.cuh", "router_gemm.cuh", "stats_update.cuh", "placement.cuh", "placement_e2r.cuh", "greedy.cuh", "sched.cuh", "host_common.h",
           "route_launch.cuh", os.path.join("..", "..", "include", "gimbal.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-Xptxas", "-v", "--expt-relaxed-constexpr"]


# extra nvcc flags for A/B builds, e.g. GIMBAL_NVCC_EXTRA=-DGIMBAL_TMA_HANDOFF=1 (part of the staleness digest)
NVCC_FLAGS += os.environ.get("GIMBAL_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _digest() -> str:
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for f in sorted(SOURCES + HEADERS):
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def stale() -> bool:
    stamp = os.path.join(OBJ, "stamp")
    if not os.path.exists(LIB) or not os.path.exists(stamp):
        return True
    return open(stamp).read().strip() != _digest()


def _compile(src: str):
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    cmd = [_nvcc()] + NVCC_FLAGS + ["-c", "-o", obj, os.path.join(CSRC, src)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return src, obj, cmd, r


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    log = []
    objs = []
    with cf.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        for src, obj, cmd, r in ex.map(_compile, SOURCES):
            log.append(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
                raise RuntimeError(f"nvcc failed on {src}")
            objs.append(obj)
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link of libgimbal.so failed")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write("\n".join(log))
    with open(os.path.join(OBJ, "stamp"), "w") as f:
        f.write(_digest())
    if verbose:
        sys.stderr.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
