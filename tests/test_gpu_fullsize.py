"""Full-size GPU parity (pytest -m gpu): BASELINE.json's configs at their real n, in the launch configuration
bench.py times (dataflow executor, bench.py's k per config), checked on sampled outputs the oracle computes one by
one (plan-order walk restricted to the sample: bit-exact) and against the fp64 reference sum (north_star
tolerances), plus the properties that hold at any size: all p outputs bitwise identical, verifier clean.
"""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import interpreter as OI
from oracle import reference as OR

pytestmark = pytest.mark.gpu

BENCH_K = {0: 8, 1: 16, 2: 8, 3: 8, 4: 8}    # bench.py's k per config


def _check_full(w, k, exec_mode, n_samples=2048, tile_units=0):
    import torch
    from paper_2606_01680_b200.device import Session
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=exec_mode, tile_units=tile_units)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    fl, sb, _, _ = B.optcc_plan_tables(plan)
    assert fl.tobytes() == oplan.flows.tobytes() and np.array_equal(sb, oplan.step_begin)
    s = Session(plan, verify=True)
    x = W.all_inputs(w)
    s.upload(x)
    s.execute()
    torch.cuda.synchronize()
    # every rank holds the same bits (PAPER.md:68 (ii)): compared on the device as raw integers
    it = torch.int32 if w.dtype == W.F32 else torch.int16
    ref = s.bufs[0].view(it)
    for r in range(1, w.p):
        assert torch.equal(ref, s.bufs[r].view(it)), f"rank {r} differs from rank 0"
    idx = W.sample_indices(w, n_samples)
    ti = torch.from_numpy(idx).to(s.device)
    ys = np.stack([s.bufs[r][ti].view(it).cpu().numpy() for r in (0, w.p - 1)])
    xs = np.ascontiguousarray(x[:, idx])
    if w.dtype == W.F32:
        ys = ys.view(np.float32)
        y_or = OI.run_f32_at(oplan, xs, idx)
        assert ys[0].tobytes() == y_or[0].tobytes() and ys[1].tobytes() == y_or[w.p - 1].tobytes()
        assert OR.check_f32(ys[0], xs).all()
    else:
        ys = ys.view(np.uint16)
        y_or = OI.run_bf16_at(oplan, xs, idx)
        assert ys[0].tobytes() == y_or[0].tobytes() and ys[1].tobytes() == y_or[w.p - 1].tobytes()
        assert OR.check_bf16(OI.bf16_bits_to_f32(ys[0]), OI.bf16_bits_to_f32(xs)).all()
    if exec_mode in (B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_COLUMN):
        # every element of every rank, device against device: the per-step executor (kernel boundaries as barriers, no
        # dependency counters, no dead-source discard) must produce the same bits as the dataflow / column executor
        plan2 = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=B.OPTCC_EXEC_PER_STEP)
        s2 = Session(plan2)
        s2.upload(x)
        s2.execute()
        torch.cuda.synchronize()
        for r in (0, w.p // 2, w.p - 1):
            assert torch.equal(s.bufs[r].view(it), s2.bufs[r].view(it)), f"executors disagree on rank {r}"
        del s2
    del x
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0 and res["checked"] == w.p * w.n
    c = B.optcc_cost(plan)
    assert c["lb_table1"] <= c["T"] * (1 + 1e-12)          # modeled T on or above the Table-1 bound
    return c


def test_c1_full_every_element():
    """configs[0] (p=4, l=2, n=2^20 f32) is small enough for the oracle to compute every element."""
    from paper_2606_01680_b200.device import Session
    w = W.config(0)
    for mode in (B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_PERSISTENT, B.OPTCC_EXEC_COLUMN):
        plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=BENCH_K[0], exec_mode=mode)
        oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=BENCH_K[0])
        x = W.all_inputs(w)
        s = Session(plan, verify=True)
        s.upload(x)
        s.execute()
        y = s.download()
        assert y.tobytes() == OI.run_f32(oplan, x).tobytes()
        assert OR.check_f32(y[0], x).all() and OR.all_ranks_identical(y)
        assert s.verify()["bad_elements"] == 0
        assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()


def test_c2_full_sampled():
    c = _check_full(W.config(1), BENCH_K[1], B.OPTCC_EXEC_DATAFLOW)
    assert c["T_over_T0"] < 1.06           # within the paper's reported gap


@pytest.mark.parametrize("tile_units", [0, 128, 1792])
@pytest.mark.parametrize("ci,k", [(1, 16), (2, 8), (3, 8), (4, 8), (1, 32), (2, 20), (3, 32)])
def test_full_sampled_column_executor(ci, k, tile_units):
    """the column executor (a tile is taken through its region's whole flow list, no synchronisation between CTAs) at
    the full sizes, with the library's tile size, warp-wide tiles (128 units) and CTA-wide tiles (1792 units): sampled
    elements against the oracle, every element against the per-step executor"""
    _check_full(W.config(ci), k, B.OPTCC_EXEC_COLUMN, n_samples=1024, tile_units=tile_units)


def test_c2_full_sampled_persistent_mode():
    _check_full(W.config(1), 4, B.OPTCC_EXEC_PERSISTENT, n_samples=512)


def test_c3_full_sampled_bf16():
    _check_full(W.config(2), BENCH_K[2], B.OPTCC_EXEC_DATAFLOW)


def test_c4_full_sampled_multi_gpu_servers():
    _check_full(W.config(3), BENCH_K[3], B.OPTCC_EXEC_DATAFLOW)


@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_COLUMN, B.OPTCC_EXEC_DATAFLOW])
@pytest.mark.parametrize("ell", W.C5_ELLS)
def test_c5_full_sampled(ell, exec_mode):
    """every ell of the C5 sweep (BASELINE.json configs[4]) at n = 2^25, through the executor bench.py times (column)
    and the dataflow executor: no straggler (C0 ring), bubble filling at 8/7, 4/3, 1.6, the Thm-1 switch 2 - 1/31,
    the algorithm's own switch ell = 2 where bubble filling turns off, and the straggler-bound regime"""
    _check_full(W.config(4, ell), BENCH_K[4], exec_mode, n_samples=1024)
