"""optcc_execute_static (include/optcc.h): optcc_execute on the library's static device workspace, for callers that
cannot allocate device memory.  Collected last on purpose (the suite runs with pytest -x).

The static entry point runs the same kernels on the same tables as optcc_execute with a caller workspace, so the bar is
the one test_gpu_parity.py uses between executors: outputs bit-identical (and, like there, bit-identical to the oracle's
plan-order emulation).  Checked on calls in a row that share the one array: the same plan twice with different inputs,
then another plan (other dtype, other executor -- its tables replace the first plan's), then the first plan again.
"""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import interpreter as OI

pytestmark = pytest.mark.gpu


def _wl(p, st, n, dtype, seed):
    ell = tuple(float(st.get(i, 1.0)) for i in range(p))
    return W.Workload(f"static{p}x{n}", p, 1, ell, n, dtype, "normal", 1.0, seed)


def _existing_path(plan, x):
    """optcc_execute with a workspace the caller allocated (device.Session)."""
    from paper_2606_01680_b200.device import Session
    s = Session(plan)
    s.upload(x)
    s.execute()
    return s.download()


def _static_path(plan, x):
    """optcc_execute_static: the rank buffers are all the device memory the caller holds."""
    import torch
    bf16 = plan.info["dtype"] == B.OPTCC_BF16
    bufs = []
    for r in range(plan.info["p"]):
        a = np.ascontiguousarray(x[r])
        t = torch.from_numpy(a.view(np.int16)).view(torch.bfloat16) if bf16 else torch.from_numpy(a)   # bit patterns
        bufs.append(t.to("cuda:0"))
    B.optcc_execute_static(plan, bufs, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    out = [(b.view(torch.int16) if bf16 else b).cpu().numpy() for b in bufs]
    return np.stack(out).view(np.uint16 if bf16 else np.float32)


def _oracle(w, k, x):
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    return OI.run_f32(oplan, x) if w.dtype == W.F32 else OI.run_bf16(oplan, x)


def test_static_workspace_matches_the_caller_workspace_path_on_calls_in_a_row():
    wa, ka = _wl(16, {0: 8.0 / 7.0}, 2 ** 17 + 2, W.F32, 501), 8        # C2 shape, several tiles and a ragged tail
    wb, kb = _wl(5, {2: 1.5}, 50003, W.BF16, 502), 4                    # bubble filling, bf16: fp32 partials in the array
    plan_a = B.optcc_plan(wa.p, wa.g, wa.ell, wa.n, wa.dtype, k=ka)     # default executor (column)
    plan_b = B.optcc_plan(wb.p, wb.g, wb.ell, wb.n, wb.dtype, k=kb, exec_mode=B.OPTCC_EXEC_DATAFLOW)
    assert plan_a.info["workspace_bytes"] <= B.OPTCC_STATIC_WORKSPACE_BYTES
    assert plan_b.info["workspace_bytes"] <= B.OPTCC_STATIC_WORKSPACE_BYTES
    calls = [(plan_a, wa, ka, W.all_inputs(wa)),
             (plan_a, wa, ka, W.all_inputs(_wl(16, {0: 8.0 / 7.0}, wa.n, W.F32, 503))),   # second call in a row, new inputs
             (plan_b, wb, kb, W.all_inputs(wb)),                                          # another plan takes the array over
             (plan_a, wa, ka, W.all_inputs(wa))]                                          # and the first one takes it back
    for plan, w, k, x in calls:
        y_static = _static_path(plan, x)
        y_ws = _existing_path(plan, x)
        assert y_static.tobytes() == y_ws.tobytes()
        assert y_static.tobytes() == _oracle(w, k, x).tobytes()
        assert all(y_static[r].tobytes() == y_static[0].tobytes() for r in range(w.p))


def test_static_workspace_rejects_plans_beyond_its_size_and_enqueues_nothing():
    import torch
    w = _wl(4, {0: 2.0}, 2 ** 20, W.BF16, 504)            # fp32 partials alone: 4 * 2^20 * 4 B = 16 MiB
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4)
    assert plan.info["workspace_bytes"] > B.OPTCC_STATIC_WORKSPACE_BYTES
    bufs = [torch.ones(w.n, dtype=torch.bfloat16, device="cuda:0") for _ in range(w.p)]
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute_static(plan, bufs)
    assert e.value.code == B.OPTCC_ETOOBIG and "ETOOBIG" in str(e.value)
    torch.cuda.synchronize()
    assert all(bool((b == 1).all()) for b in bufs)        # the rank buffers are untouched


def test_static_workspace_holds_the_metric_config_at_full_size():
    """BASELINE config 1 (C2: p = 16, n = 2^26 fp32, bench.py's k = 16) is the largest plan the 8 MiB array is sized for;
    outputs compared on the device with the caller-workspace path, bit for bit, on two calls in a row."""
    import torch
    from paper_2606_01680_b200.device import Session
    w = W.config(1)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=16)
    assert plan.info["workspace_bytes"] <= B.OPTCC_STATIC_WORKSPACE_BYTES
    s = Session(plan)
    g = torch.Generator(device="cuda:0").manual_seed(505)
    for _ in range(2):
        x = [torch.randn(w.n, dtype=torch.float32, device="cuda:0", generator=g) for _ in range(w.p)]
        for r in range(w.p):
            s.bufs[r].copy_(x[r])
        s.execute()
        B.optcc_execute_static(plan, x, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert all(torch.equal(x[r].view(torch.int32), s.bufs[r].view(torch.int32)) for r in range(w.p))
        assert torch.equal(x[0].view(torch.int32), x[w.p - 1].view(torch.int32))
