"""TEST INFRASTRUCTURE ONLY: builds oracle/walk.c (gcc) and calls it.  The C walk is interpreter.run_f32 restated --
same table, same order, same one-add-per-element arithmetic -- and is pinned against it bit for bit
(tests/test_oracle_cwalk.py).  bench.py's cpu_baseline times it beside the numpy walk; nothing in the product imports it.
"""
import ctypes as C
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "walk.c")
LIB = os.path.join(HERE, "liboraclewalk.so")
_lib = None


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("gcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


def load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(LIB)
        lib.oracle_walk_f32.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_uint32]
        lib.oracle_walk_f32.restype = C.c_int
        lib.oracle_walk_threads.restype = C.c_int
        _lib = lib
    return _lib


def threads():
    return int(load().oracle_walk_threads())


def run_f32(plan, x, copy=True):
    """plan: oracle.planner.Plan (fp32); x[p, n] float32.  Returns the p outputs [p, n] (in place if copy=False)."""
    y = np.array(x, dtype=np.float32, copy=True, order="C") if copy else x
    assert y.dtype == np.float32 and y.flags["C_CONTIGUOUS"] and y.shape == (plan.p, plan.n)
    flows = np.ascontiguousarray(plan.flows)
    sb = np.ascontiguousarray(plan.step_begin, dtype=np.uint32)
    assert flows.dtype.itemsize == 40 and len(sb) == plan.n_steps + 1
    rc = load().oracle_walk_f32(y.ctypes.data, plan.p, plan.n, flows.ctypes.data, sb.ctypes.data, plan.n_steps)
    if rc != 0:
        raise ValueError("oracle_walk_f32: a flow record is out of range")
    return y
