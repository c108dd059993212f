"""Builds liboptcc.so (C-ABI library: host planner + cost model + sm_100a executor) in-tree with nvcc.

    python -m paper_2606_01680_b200.build [--force]

nvcc cross-compiles for sm_100a without a GPU.  The library links the static CUDA runtime, so it loads on a
box without a driver; only the execute / verify entry points need a device.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liboptcc.so")
SOURCES = ["optcc_plan.cpp", "optcc_cost.cpp", "optcc_exec.cu"]
HEADERS = [os.path.join(ROOT, "include", "optcc.h"), os.path.join(CSRC, "optcc_internal.h"),
           os.path.join(CSRC, "optcc_kernels.cuh")]


def _nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: liboptcc cannot be built (there is no CPU fallback)")
    return exe


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), "-shared", "-o", LIB, "-std=c++17", "-O3", "-lineinfo",
           "-gencode", "arch=compute_100a,code=sm_100a",
           "-Xcompiler", "-fPIC,-pthread,-ffp-contract=off,-fvisibility=hidden,-Wall",
           "-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
