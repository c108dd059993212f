"""Thin ctypes binding over liboptcc.so (include/optcc.h).  Argument marshalling only: every step of the
path (planning, costing, executing, verifying) runs inside the C-ABI library.  Function names mirror the C ones.

There is no fallback: if liboptcc.so is missing, `load()` raises (build it with
`python -m paper_2606_01680_b200.build` or `__graft_entry__.build()`).
Device pointers are passed as Python ints or as objects with `.data_ptr()` (torch tensors); torch itself is
not imported here.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liboptcc.so")

OPTCC_F32, OPTCC_BF16 = 0, 1
OPTCC_OK, OPTCC_EINVAL, OPTCC_EUNSUPPORTED, OPTCC_ENOMEM, OPTCC_ECUDA, OPTCC_EVERIFY, OPTCC_ESTALE, OPTCC_ETOOBIG = range(8)
OPTCC_STATIC_WORKSPACE_BYTES = 8 << 20   # include/optcc.h
OPTCC_EXEC_AUTO, OPTCC_EXEC_PERSISTENT, OPTCC_EXEC_PER_STEP, OPTCC_EXEC_DATAFLOW, OPTCC_EXEC_COLUMN = 0, 1, 2, 3, 4
EXEC_NAMES = {0: "auto", 1: "persistent", 2: "per_step", 3: "dataflow", 4: "column"}
OPTCC_SCHED_OPTCC, OPTCC_SCHED_RING_DEGRADED = 0, 1
ERROR_NAMES = {1: "EINVAL", 2: "EUNSUPPORTED", 3: "ENOMEM", 4: "ECUDA", 5: "EVERIFY", 6: "ESTALE", 7: "ETOOBIG"}

# optcc_flow_t (PLAN_SPEC 3): 40 bytes
FLOW_DTYPE = np.dtype([
    ("off", "<u8"), ("len", "<u8"), ("step", "<u4"), ("seg", "<u4"), ("sec", "<u4"),
    ("src", "<u2"), ("dst", "<u2"), ("op", "u1"), ("stage", "u1"), ("link", "u1"), ("part", "u1"),
    ("reserved", "<u4"),
], align=False)


class optcc_opts_t(C.Structure):
    _fields_ = [("k", C.c_uint32), ("exec_mode", C.c_uint32), ("grid_ctas", C.c_uint32), ("copy_path", C.c_uint32),
                ("step_limit", C.c_uint32), ("tile_units", C.c_uint32), ("schedule", C.c_uint32), ("ordering", C.c_uint32), ("no_discard", C.c_uint32), ("verify_eager", C.c_uint32),
                ("col_order", C.c_uint32), ("no_forward", C.c_uint32), ("reserved", C.c_uint32 * 4)]


class optcc_plan_info_t(C.Structure):
    _fields_ = [(n, C.c_uint32) for n in ("p", "g", "q", "m", "H", "k", "construction", "dtype", "unit_elems", "mask_words")] + \
               [(n, C.c_uint64) for n in ("n", "n_ring", "n_p2p", "U", "U_ring", "U_p2p")] + \
               [(n, C.c_uint32) for n in ("n_steps", "n_flows", "max_flows_per_step", "n_sec_bounds", "n_p2p_bounds", "mask_bytes")] + \
               [(n, C.c_uint64) for n in ("reduce_elems", "copy_elems", "workspace_bytes", "verify_workspace_bytes",
                                          "mask_offset_bytes", "padded_n")] + \
               [("plan_build_seconds", C.c_double), ("lazy_verify", C.c_uint32), ("exec_mode", C.c_uint32)]


class optcc_cost_params_t(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("alpha_latency", C.c_double), ("sync", C.c_double)]


class optcc_cost_t(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("T", "T0", "T_over_T0", "T_closed_form", "T_limit", "lb_table1", "lb_tight",
                                          "T0_server", "bodies", "straggler_sent", "straggler_recv", "T_ring_degraded", "T_r2ccl")] + \
               [(n, C.c_int32) for n in ("lb_table1_thm", "lb_tight_thm", "regime", "reserved")]


class optcc_verify_result_t(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("bad_elements", "overlap_elements", "first_bad", "checked")]


class OptccError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        self.name = ERROR_NAMES.get(code, str(code))
        super().__init__(f"{what}: {self.name} ({load().optcc_strerror(code).decode()})"
                         + (f", cudaError {load().optcc_last_cuda_error()}" if code == OPTCC_ECUDA else ""))


_lib = None
EXPORTS = ("optcc_plan", "optcc_plan_ex", "optcc_plan_destroy", "optcc_plan_info", "optcc_plan_tables", "optcc_cost",
           "optcc_prepare", "optcc_column_tables", "optcc_execute", "optcc_execute_static", "optcc_execute_shard", "optcc_verify_shard", "optcc_peer_alloc", "optcc_peer_open", "optcc_peer_close", "optcc_peer_free", "optcc_execute_host", "optcc_execute_host_sharded", "optcc_workspace_check", "optcc_workspace_forget",
           "optcc_verify", "optcc_strerror",
           "optcc_last_cuda_error", "optcc_abi_version")


def load():
    """dlopen liboptcc.so and declare the prototypes of include/optcc.h.  Raises if the library is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it (python -m paper_2606_01680_b200.build). "
                           "There is no CPU or PyTorch fallback for the OPTCC executor.")
    lib = C.CDLL(LIB_PATH)
    vp, u64 = C.c_void_p, C.c_uint64
    lib.optcc_plan.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), u64, C.c_int, C.POINTER(vp)]
    lib.optcc_plan_ex.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), u64, C.c_int, C.POINTER(optcc_opts_t), C.POINTER(vp)]
    lib.optcc_plan_destroy.argtypes = [vp]
    lib.optcc_plan_destroy.restype = None
    lib.optcc_plan_info.argtypes = [vp, C.POINTER(optcc_plan_info_t)]
    lib.optcc_plan_tables.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    lib.optcc_cost.argtypes = [vp, C.POINTER(optcc_cost_params_t), C.POINTER(optcc_cost_t)]
    lib.optcc_prepare.argtypes = [vp, vp, vp]
    lib.optcc_column_tables.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_uint32), C.POINTER(vp), C.POINTER(C.c_uint32)]
    lib.optcc_execute.argtypes = [vp, C.POINTER(vp), vp, vp]
    lib.optcc_execute_static.argtypes = [vp, C.POINTER(vp), vp]
    lib.optcc_execute_shard.argtypes = [vp, C.POINTER(vp), vp, vp, C.c_uint32, C.c_uint32]
    lib.optcc_verify_shard.argtypes = [vp, vp, vp, C.c_uint32, C.c_uint32, C.POINTER(optcc_verify_result_t)]
    lib.optcc_peer_alloc.argtypes = [u64, C.POINTER(vp), C.c_char_p]
    lib.optcc_peer_open.argtypes = [C.c_char_p, C.POINTER(vp)]
    lib.optcc_peer_close.argtypes = [vp]
    lib.optcc_peer_free.argtypes = [vp]
    lib.optcc_execute_host.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), vp, vp]
    lib.optcc_execute_host_sharded.argtypes = [vp, u64, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), vp, vp]
    lib.optcc_verify.argtypes = [vp, vp, vp, C.POINTER(optcc_verify_result_t)]
    lib.optcc_workspace_check.argtypes = [vp, vp, vp]
    lib.optcc_workspace_forget.argtypes = [vp]
    lib.optcc_workspace_forget.restype = None
    lib.optcc_strerror.argtypes = [C.c_int]
    lib.optcc_strerror.restype = C.c_char_p
    lib.optcc_last_cuda_error.argtypes = []
    lib.optcc_abi_version.argtypes = []
    for name in EXPORTS:
        if name not in ("optcc_plan_destroy", "optcc_strerror", "optcc_workspace_forget"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ptr(x):
    if x is None:
        return None
    return int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x)


def _ptr_array(xs):
    arr = (C.c_void_p * len(xs))()
    for i, x in enumerate(xs):
        arr[i] = _ptr(x)
    return arr


def _struct_dict(s):
    return {name: getattr(s, name) for name, _ in s._fields_}


class Plan:
    """Owns one optcc_plan_t*.  `info` is a dict of optcc_plan_info_t."""

    def __init__(self, handle):
        self._h = C.c_void_p(handle)
        info = optcc_plan_info_t()
        rc = load().optcc_plan_info(self._h, C.byref(info))
        if rc:
            raise OptccError(rc, "optcc_plan_info")
        self.info = _struct_dict(info)

    @property
    def handle(self):
        if not self._h:
            raise RuntimeError("plan destroyed")
        return self._h

    def destroy(self):
        if self._h:
            load().optcc_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def optcc_plan(p, g, ell, n, dtype, k=0, exec_mode=OPTCC_EXEC_AUTO, grid_ctas=0, copy_path=0, step_limit=0, tile_units=0, schedule=0, ordering=0, no_discard=0, verify_eager=0, col_order=0, no_forward=0):
    """optcc_plan_ex: returns a Plan.  ell: sequence of p floats."""
    lib = load()
    ell_arr = (C.c_double * len(ell))(*[float(x) for x in ell])
    opts = optcc_opts_t(k, exec_mode, grid_ctas, copy_path, step_limit, tile_units, schedule, ordering, no_discard, verify_eager, col_order, no_forward)
    h = C.c_void_p()
    rc = lib.optcc_plan_ex(int(p), int(g), ell_arr, int(n), int(dtype), C.byref(opts), C.byref(h))
    if rc:
        raise OptccError(rc, "optcc_plan")
    return Plan(h.value)


def optcc_plan_tables(plan):
    """Copies of the borrowed host tables: (flows[FLOW_DTYPE], step_begin[u32], sec_bounds[u64], p2p_bounds[u64])."""
    f, sb, sec, p2p = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
    rc = load().optcc_plan_tables(plan.handle, C.byref(f), C.byref(sb), C.byref(sec), C.byref(p2p))
    if rc:
        raise OptccError(rc, "optcc_plan_tables")
    i = plan.info

    def view(ptr, count, dt):
        if count == 0 or not ptr.value:
            return np.zeros(0, dtype=dt)
        buf = (C.c_char * (count * np.dtype(dt).itemsize)).from_address(ptr.value)
        return np.frombuffer(buf, dtype=dt, count=count).copy()

    return (view(f, i["n_flows"], FLOW_DTYPE), view(sb, i["n_steps"] + 1, np.uint32),
            view(sec, i["n_sec_bounds"], np.uint64), view(p2p, i["n_p2p_bounds"], np.uint64))


# the column executor's record (optcc.h: optcc_column_tables): 32 bytes
COLREC_DTYPE = np.dtype([("off", "<u8"), ("len", "<u8"), ("src", "<u2"), ("dst", "<u2"), ("op", "u1"), ("ksrc", "u1"),
                         ("kdin", "u1"), ("kdout", "u1"), ("flags", "<u4"), ("pad", "<u4")], align=False)
COLITEM_DTYPE = np.dtype([("first", "<u4"), ("end", "<u4"), ("tile", "<u4"), ("units", "<u4")], align=False)


def optcc_column_tables(plan):
    """Copies of the column executor's host tables: (records[COLREC_DTYPE], items[COLITEM_DTYPE]).  No device needed."""
    rec, it = C.c_void_p(), C.c_void_p()
    nrec, nit = C.c_uint32(), C.c_uint32()
    rc = load().optcc_column_tables(plan.handle, C.byref(rec), C.byref(nrec), C.byref(it), C.byref(nit))
    if rc:
        raise OptccError(rc, "optcc_column_tables")

    def view(ptr, count, dt):
        if count == 0 or not ptr.value:
            return np.zeros(0, dtype=dt)
        buf = (C.c_char * (count * np.dtype(dt).itemsize)).from_address(ptr.value)
        return np.frombuffer(buf, dtype=dt, count=count).copy()

    return view(rec, nrec.value, COLREC_DTYPE), view(it, nit.value, COLITEM_DTYPE)


def optcc_cost(plan, alpha=0.0, beta=1.0, alpha_latency=0.0, sync=0.0):
    out = optcc_cost_t()
    params = optcc_cost_params_t(alpha, beta, alpha_latency, sync)
    rc = load().optcc_cost(plan.handle, C.byref(params), C.byref(out))
    if rc:
        raise OptccError(rc, "optcc_cost")
    return _struct_dict(out)


def optcc_prepare(plan, workspace, stream=None):
    rc = load().optcc_prepare(plan.handle, _ptr(workspace), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_prepare")


def optcc_execute(plan, bufs, workspace, stream=None):
    """bufs: p device buffers (torch tensors or ints).  Asynchronous on `stream` (a cudaStream_t as int)."""
    rc = load().optcc_execute(plan.handle, _ptr_array(bufs), _ptr(workspace), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_execute")


def optcc_execute_static(plan, bufs, stream=None):
    """optcc_execute on the library's static device workspace (no device allocation; plans up to
    OPTCC_STATIC_WORKSPACE_BYTES of workspace, else OptccError ETOOBIG)."""
    rc = load().optcc_execute_static(plan.handle, _ptr_array(bufs), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_execute_static")


def optcc_execute_shard(plan, bufs, workspace, shard, n_shards, stream=None):
    """The work items i = shard (mod n_shards) of the plan; bufs may be peer-mapped pointers (see peers.py)."""
    rc = load().optcc_execute_shard(plan.handle, _ptr_array(bufs), _ptr(workspace), _ptr(stream), int(shard), int(n_shards))
    if rc:
        raise OptccError(rc, "optcc_execute_shard")


def optcc_verify_shard(plan, workspace, shard, n_shards, stream=None, raise_on_fail=True):
    out = optcc_verify_result_t()
    rc = load().optcc_verify_shard(plan.handle, _ptr(workspace), _ptr(stream), int(shard), int(n_shards), C.byref(out))
    if rc and (rc != OPTCC_EVERIFY or raise_on_fail):
        raise OptccError(rc, "optcc_verify_shard")
    return _struct_dict(out)


def optcc_peer_alloc(nbytes):
    """-> (device pointer, 64-byte handle other processes can open)"""
    ptr = C.c_void_p()
    handle = C.create_string_buffer(64)
    rc = load().optcc_peer_alloc(int(nbytes), C.byref(ptr), handle)
    if rc:
        raise OptccError(rc, "optcc_peer_alloc")
    return ptr.value, handle.raw


def optcc_peer_open(handle):
    ptr = C.c_void_p()
    rc = load().optcc_peer_open(C.create_string_buffer(bytes(handle), 64), C.byref(ptr))
    if rc:
        raise OptccError(rc, "optcc_peer_open")
    return ptr.value


def optcc_peer_close(ptr):
    rc = load().optcc_peer_close(int(ptr))
    if rc:
        raise OptccError(rc, "optcc_peer_close")


def optcc_peer_free(ptr):
    rc = load().optcc_peer_free(int(ptr))
    if rc:
        raise OptccError(rc, "optcc_peer_free")


def optcc_execute_host(plan, host_in, host_out, bufs, workspace, stream=None):
    rc = load().optcc_execute_host(plan.handle, _ptr_array(host_in), _ptr_array(host_out), _ptr_array(bufs),
                                   _ptr(workspace), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_execute_host")


def optcc_execute_host_sharded(plan, n_total, host_in, host_out, bufs, workspace, stream=None):
    """n_total / plan.n element shards, all with `plan`; H2D, execution and D2H of neighbouring shards overlap."""
    rc = load().optcc_execute_host_sharded(plan.handle, int(n_total), _ptr_array(host_in), _ptr_array(host_out),
                                           _ptr_array(bufs), _ptr(workspace), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_execute_host_sharded")


def optcc_workspace_check(plan, workspace, stream=None):
    """Synchronises `stream`; raises OptccError (ESTALE) if a launch did not find this plan's tables in the workspace."""
    rc = load().optcc_workspace_check(plan.handle, _ptr(workspace), _ptr(stream))
    if rc:
        raise OptccError(rc, "optcc_workspace_check")


def optcc_workspace_forget(workspace):
    load().optcc_workspace_forget(_ptr(workspace))


def optcc_verify(plan, workspace, stream=None, raise_on_fail=True):
    out = optcc_verify_result_t()
    rc = load().optcc_verify(plan.handle, _ptr(workspace), _ptr(stream), C.byref(out))
    if rc and (rc != OPTCC_EVERIFY or raise_on_fail):
        raise OptccError(rc, "optcc_verify")
    return _struct_dict(out)
