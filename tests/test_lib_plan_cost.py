"""CPU tests of liboptcc's host side (no GPU): the library loads and exports every symbol of include/optcc.h;
the C++ planner's integer tables equal the oracle's byte for byte (north_star: "integer plan/step tables match
bit-exactly"); optcc_cost agrees with the oracle's exact-rational simulation and closed forms to 1e-12 relative.
"""
import math
import os
import re

import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import build as optcc_build
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import cost_sim, closed_forms as cf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    optcc_build.build()


def _ell(p, d):
    return [float(d.get(i, 1.0)) for i in range(p)]


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "optcc.h")).read()
    declared = set(re.findall(r"OPTCC_API\s+[\w\s\*]+?\b(optcc_\w+)\s*\(", header))
    assert declared == set(B.EXPORTS)
    lib = B.load()
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.optcc_abi_version() == 2
    assert B.FLOW_DTYPE.itemsize == 40


def _compare(p, g, ell, n, dtype, k):
    pl = B.optcc_plan(p, g, ell, n, dtype, k=k)
    op = OP.build_plan(p, g, list(ell), n, dtype, k=k)
    fl, sb, sec, p2p = B.optcc_plan_tables(pl)
    i = pl.info
    assert fl.tobytes() == op.flows.tobytes()
    assert np.array_equal(sb, op.step_begin)
    assert np.array_equal(sec, op.sec_bounds)
    assert np.array_equal(p2p, op.p2p_bounds)
    for key, val in (("p", op.p), ("g", op.g), ("q", op.q), ("m", op.m), ("H", op.H), ("k", op.k),
                     ("construction", op.construction), ("unit_elems", op.A), ("n", op.n), ("n_ring", op.n_ring),
                     ("n_p2p", op.n_p2p), ("U", op.U), ("U_ring", op.U_ring), ("U_p2p", op.U_p2p),
                     ("n_steps", op.n_steps), ("n_flows", len(op.flows))):
        assert i[key] == val, key
    assert i["reduce_elems"] == (p - 1) * n and i["copy_elems"] == (p - 1) * n   # Lemma 4 with equality (:340)
    return pl, op


@pytest.mark.parametrize("ci", range(5))
@pytest.mark.parametrize("k", [0, 8])
def test_tables_equal_oracle_on_baseline_configs(ci, k):
    w = W.config(ci)
    _compare(w.p, w.g, w.ell, w.n, w.dtype, k)


@pytest.mark.parametrize("ell", W.C5_ELLS)
def test_tables_equal_oracle_on_c5_sweep(ell):
    w = W.config(4, ell)
    _compare(w.p, w.g, w.ell, w.n, w.dtype, 0)


GRID = [
    # p, g, stragglers, n, dtype, k
    (3, 1, {0: 2.0}, 1, 0, 4), (3, 1, {1: 1.5}, 7, 0, 4), (4, 1, {}, 1001, 0, 0), (5, 1, {0: 2.0}, 4803, 0, 4),
    (5, 1, {2: 1.5}, 4803, 1, 4), (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 10007, 0, 4), (7, 1, {3: 1.25, 6: 1.25}, 99991, 1, 8),
    (16, 1, {9: 8.0 / 7.0}, 123457, 0, 8), (12, 4, {4: 2.0, 5: 2.0, 6: 2.0, 7: 2.0}, 65537, 0, 4),
    (12, 2, {0: 1.5, 1: 1.5}, 4097, 1, 12), (32, 1, {0: 2.0 - 1.0 / 31.0}, 1 << 20, 0, 20), (32, 1, {31: 3.0}, 999983, 1, 0),
    (9, 3, {3: 8.0 / 7.0, 4: 8.0 / 7.0, 5: 8.0 / 7.0}, 30011, 0, 8), (6, 1, {1: 1.0 + 2 ** -40}, 5000, 0, 4),
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 70001, 1, 4), (40, 8, {r: 2.0 for r in range(8, 16)}, 262147, 0, 8),
    (12, 2, {0: 2.0, 1: 2.0, 6: 1.5, 7: 1.5}, 30011, 0, 4),          # g > 1 with two straggler servers (composed C3)
    (32, 4, {**{r: 2.0 for r in range(4, 8)}, **{r: 8.0 / 7.0 for r in range(20, 24)}, **{r: 2.0 for r in range(28, 32)}}, 100003, 1, 8),
]


@pytest.mark.parametrize("p,g,st,n,dtype,k", GRID)
def test_tables_equal_oracle_on_grid(p, g, st, n, dtype, k):
    _compare(p, g, _ell(p, st), n, dtype, k)


@pytest.mark.parametrize("args,code", [
    ((2, 1, [1.0, 2.0], 10, 0, 0), "EINVAL"),                 # p >= 3 (:68)
    ((4, 3, [1.0] * 4, 10, 0, 0), "EINVAL"),                  # g | p
    ((4, 1, [1.0, 0.5, 1.0, 1.0], 10, 0, 0), "EINVAL"),       # ell >= 1
    ((4, 1, [1.0, float("nan"), 1.0, 1.0], 10, 0, 0), "EINVAL"),
    ((4, 2, [1.0, 2.0, 1.0, 1.0], 10, 0, 0), "EINVAL"),       # one ell per server (:274)
    ((4, 1, [2.0, 2.0, 2.0, 1.0], 10, 0, 0), "EINVAL"),       # two healthy servers needed
    ((4, 1, [2.0, 1.0, 1.0, 1.0], 0, 0, 0), "EINVAL"),        # n > 0
    ((4, 1, [2.0, 1.0, 1.0, 1.0], 10, 0, 6), "EINVAL"),       # k multiple of 4 (:155)
    ((4, 1, [2.0, 1.0, 1.0, 1.0], 10, 7, 0), "EINVAL"),       # dtype
    ((8, 2, [1.0] * 8, 10, 0, 0), "EUNSUPPORTED"),
])
def test_error_codes_match_oracle(args, code):
    p, g, ell, n, dtype, k = args
    with pytest.raises(OP.PlanError) as eo:
        OP.build_plan(p, g, ell, n, dtype, k=k)
    assert eo.value.code == code
    with pytest.raises(B.OptccError) as el:
        B.optcc_plan(p, g, ell, n, dtype, k=k)
    assert el.value.name == code


COST_CASES = [
    (4, 1, {0: 2.0}, 4 * 3 * 8 * 16, 0, 8), (5, 1, {0: 1.5}, 4 * 4 * 4 * 50, 0, 4), (16, 1, {0: 8.0 / 7.0}, 1 << 16, 0, 8),
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 4 * 5 * 8 * 9, 0, 8), (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 8 * 61 * 8 * 3, 1, 8),
    (16, 4, {r: 2.0 for r in range(4)}, 4 * 4 * 3 * 8 * 5, 0, 8), (32, 1, {0: 3.0}, 4 * 31 * 12 * 7, 0, 12),
    (6, 1, {}, 6000, 0, 0), (12, 2, {0: 1.5, 1: 1.5}, 4097, 1, 12),
]


@pytest.mark.parametrize("p,g,st,n,dtype,k", COST_CASES)
def test_cost_matches_oracle_simulation_and_closed_forms(p, g, st, n, dtype, k):
    ell = _ell(p, st)
    pl, op = _compare(p, g, ell, n, dtype, k)
    c = B.optcc_cost(pl)
    sim = cost_sim.simulate(op)
    lbs = cost_sim.lower_bounds(op)
    rel = lambda a, b: abs(a - float(b)) <= 1e-12 * abs(float(b))
    assert rel(c["T"], sim["T"])
    assert rel(c["T0"], sim["T0"])
    assert rel(c["T_over_T0"], sim["ratio"])
    assert rel(c["lb_table1"], lbs["table1"])
    if lbs["tight"] is None:
        assert math.isnan(c["lb_tight"])
    else:
        assert rel(c["lb_tight"], lbs["tight"])
    assert rel(c["T_closed_form"], cost_sim.paper_closed_form(op))
    assert rel(c["T0_server"], cf.T0_server(p, n, g))
    assert c["T"] >= c["lb_table1"] * (1 - 1e-12)
    if op.m:
        r = op.stragglers[0] * g
        assert c["straggler_sent"] == sim["nic_sent"][r] and c["straggler_recv"] == sim["nic_recvd"][r]
    # alpha-beta: a fixed cost per flow and a scaled element time
    c2 = B.optcc_cost(pl, alpha=0.25, beta=3.0)
    sim2 = cost_sim.simulate(op, alpha=cf.Fr(1, 4), beta=3)
    assert rel(c2["T"], sim2["T"])


def test_cost_reports_paper_numbers_for_baseline_configs(golden):
    """Modeled T/T0 lies on or above the Table-1 bound and within the paper's reported gap (north_star)."""
    w = W.config(1)                       # C2: Eq.(2) exact for the canonical plan (:185)
    pl = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=20)
    c = B.optcc_cost(pl)
    assert c["lb_table1"] <= c["T"]
    assert abs(c["T"] / c["T_closed_form"] - 1) < 1e-5       # n not divisible by k(p-1): unit rounding only
    assert c["T_over_T0"] < 1.06                               # "within 2-6 %" (:7, :217)
    w = W.config(0)                       # C1: l = 2, T/T0 -> 4/3 (k+1)/k
    c = B.optcc_cost(B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=8))
    assert abs(c["T_over_T0"] - (4.0 / 3.0) * 9 / 8) < 1e-4       # 2^20 is not divisible by 3k: unit rounding
    assert c["regime"] == 2 and c["lb_table1_thm"] == 1 and c["lb_tight_thm"] == 6


def test_plan_build_time_is_submillisecond_scale_at_p1024():
    """schedule generation '< 1 ms at p=1024' is for closed-form rules; ours also materialises and
    sorts every flow, so only a loose bound is asserted, the measured value is reported by bench.py."""
    p = 1024
    pl = B.optcc_plan(p, 1, _ell(p, {0: 2.0}), 1 << 26, 0, k=4)
    assert pl.info["n_flows"] > 0
    assert pl.info["plan_build_seconds"] < 5.0


@pytest.mark.parametrize("ci,ell,k,gap", [
    (0, None, 32, 1.06), (1, None, 20, 1.06), (2, None, 20, 1.085), (3, None, 32, 1.06),
    (4, 1.0, 20, 1.06), (4, 8.0 / 7.0, 20, 1.06), (4, 4.0 / 3.0, 20, 1.06), (4, 1.6, 20, 1.06),
    (4, 2.0 - 1.0 / 31.0, 20, 1.06), (4, 2.0, 20, 1.06), (4, 3.0, 20, 1.06),
])
def test_modeled_time_within_the_papers_gap_on_every_config(ci, ell, k, gap):
    """north_star: 'modeled T/T0 lies on or above the Table 1 lower bound and within the paper's reported gap'
    (<= 6 % single straggler :217, <= 8.5 % multi-straggler :219, <= 6 % multi-GPU) at the k SURVEY 8(d) names."""
    w = W.config(ci, ell) if ci == 4 else W.config(ci)
    c = B.optcc_cost(B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k))
    assert c["lb_table1"] <= c["T"] * (1 + 1e-12)
    lb = c["lb_table1"] if math.isnan(c["lb_tight"]) else c["lb_tight"]
    assert c["T"] / lb <= gap
    assert c["T"] <= c["T_closed_form"] * (1 + 1e-3)      # never above the paper's own finite-k form (up to unit rounding)


@pytest.mark.parametrize("ci,k", [(0, 8), (1, 16), (2, 8), (3, 8), (4, 8)])
def test_column_executor_plans_are_the_same_tables(ci, k):
    """exec_mode only selects the executor: the plan tables, the cost and the mask layout of a column-executor plan are
    those of the default plan; its workspace additionally holds one work item per (region, tile)."""
    from paper_2606_01680_b200 import workloads as W
    w = W.config(ci)
    n = min(w.n, 2 ** 20)
    a = B.optcc_plan(w.p, w.g, w.ell, n, w.dtype, k=k)
    b = B.optcc_plan(w.p, w.g, w.ell, n, w.dtype, k=k, exec_mode=B.OPTCC_EXEC_COLUMN)
    ta, tb = B.optcc_plan_tables(a), B.optcc_plan_tables(b)
    for x, y in zip(ta, tb):
        assert np.asarray(x).tobytes() == np.asarray(y).tobytes()
    ia, ib = a.info, b.info
    for key in ("n_steps", "n_flows", "k", "mask_bytes", "lazy_verify", "padded_n", "reduce_elems", "copy_elems"):
        assert ia[key] == ib[key]
    assert ib["workspace_bytes"] % 256 == 0 and ib["verify_workspace_bytes"] >= ib["workspace_bytes"]
    assert B.optcc_cost(a)["T"] == B.optcc_cost(b)["T"]


# ---- latency-type fixed cost and sync messages (PLAN_SPEC 6; PAPER.md:201 fn.5, :199, :217) ----
@pytest.mark.parametrize("p", [3, 4, 8, 16, 33])
def test_latency_alpha_on_the_fault_free_ring_is_the_textbook_alpha_beta_time(p):
    """The fault-free ring with a latency-type alpha: T = 2(p-1)(n/p beta + alpha) -- the alpha-beta model of a ring
    AllReduce (the closed form the 86 % / 14 % split of PAPER.md:201 fn.5 is calibrated on) -- as an equality of
    rationals in the oracle, and 1e-12 in the library."""
    from fractions import Fraction as Fr
    n = 4 * p * 250
    oplan = OP.build_plan(p, 1, [1.0] * p, n, OP.F32)
    al, beta = Fr(7, 3), Fr(5, 4)
    sim = cost_sim.simulate(oplan, beta=beta, alpha_latency=al)
    assert sim["T"] == 2 * (p - 1) * (Fr(n, p) * beta + al)
    c = B.optcc_cost(B.optcc_plan(p, 1, [1.0] * p, n, B.OPTCC_F32), beta=float(beta), alpha_latency=float(al))
    assert abs(c["T"] - float(sim["T"])) <= 1e-12 * float(sim["T"])
    # calibrated to 14 % fixed overhead: alpha = (0.14 / 0.86) n beta / p  =>  bandwidth share of T is exactly 86 %
    al = Fr(14, 86) * Fr(n, p) * beta
    sim = cost_sim.simulate(oplan, beta=beta, alpha_latency=al)
    assert cf.T0(p, n, 1) * beta / sim["T"] == Fr(86, 100)


@pytest.mark.parametrize("p,g,st,n,k,kw", [
    (5, 1, {0: 2.0}, 4 * 4 * 4 * 25, 4, {}), (16, 1, {3: 8.0 / 7.0}, 123456, 8, {}), (9, 1, {1: 1.5}, 99999, 12, {"ordering": 3}),
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 65539, 4, {}), (16, 4, {r: 2.0 for r in range(4)}, 40001, 4, {}), (6, 1, {}, 7777, 0, {}),
])
def test_latency_alpha_and_sync_agree_with_the_oracles_rationals(p, g, st, n, k, kw):
    from fractions import Fraction as Fr
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    oplan = OP.build_plan(p, g, ell, n, OP.F32, k=k, **kw)
    plan = B.optcc_plan(p, g, ell, n, B.OPTCC_F32, k=k, **kw)
    base = cost_sim.simulate(oplan)
    prev = base["T"]
    for al, sy, a_occ in ((Fr(0), Fr(0), Fr(0)), (Fr(37, 2), Fr(0), Fr(0)), (Fr(37, 2), Fr(5, 4), Fr(0)), (Fr(1000), Fr(3), Fr(1, 4))):
        sim = cost_sim.simulate(oplan, alpha=a_occ, alpha_latency=al, sync=sy)
        c = B.optcc_cost(plan, alpha=float(a_occ), alpha_latency=float(al), sync=float(sy))
        assert abs(c["T"] - float(sim["T"])) <= 1e-12 * float(sim["T"])
        assert sim["T"] >= prev                      # fixed costs never speed a plan up
        prev = sim["T"]
    assert cost_sim.simulate(oplan, alpha_latency=0, sync=0)["T"] == base["T"]


def test_a_latency_shorter_than_a_slot_is_hidden_by_the_neighbouring_stage():
    """What makes the fixed cost a latency and not an occupancy: in the canonical plan a ring link
    carries Stage 1 of one segment and Stage 4 of another back to back, so a chain's next hop starts one slot after the
    previous one ended; a latency up to one slot only delays the drain of the pipeline, an occupancy of the same size
    is paid in every one of the (k+1)(p-1) windows."""
    from fractions import Fraction as Fr
    p, k = 9, 8
    n = 4 * (p - 1) * k * 50
    ell = [1.0] * p
    ell[0] = 2.0
    oplan = OP.build_plan(p, 1, ell, n, OP.F32, k=k)
    s = Fr(n, k * (p - 1))                                   # one slot
    base = cost_sim.simulate(oplan)["T"]
    lat = cost_sim.simulate(oplan, alpha_latency=s / 2)["T"]
    occ = cost_sim.simulate(oplan, alpha=s / 2)["T"]
    assert lat - base <= 2 * (p - 1) * (s / 2)               # at most one latency per hop of the last segment's chains
    assert occ - base >= (k + 1) * (p - 1) * (s / 2)         # one occupancy per window


def test_entry_points_reject_bad_arguments_before_touching_a_device():
    """Argument checks that need no GPU: optcc_execute_static refuses a plan whose workspace exceeds the static array
    (OPTCC_ETOOBIG) and optcc_execute_shard / optcc_verify_shard refuse a shard out of range (EINVAL) or a plan whose
    executor has no independent work items (EUNSUPPORTED) -- all before the first CUDA call, so this runs on a CPU box."""
    import ctypes as C
    lib = B.load()
    p, n = 4, 2 ** 20
    ell = [2.0, 1.0, 1.0, 1.0]
    big = B.optcc_plan(p, 1, ell, n, W.BF16, k=4)                       # fp32 partials alone: 16 MiB
    assert big.info["workspace_bytes"] > B.OPTCC_STATIC_WORKSPACE_BYTES
    fake = (C.c_void_p * p)(*[0x1000 * (i + 1) for i in range(p)])      # never dereferenced
    assert lib.optcc_execute_static(big.handle, fake, None) == B.OPTCC_ETOOBIG
    assert b"OPTCC_STATIC_WORKSPACE_BYTES" in lib.optcc_strerror(B.OPTCC_ETOOBIG)
    small = B.optcc_plan(p, 1, ell, 4096, W.F32, k=4)
    assert small.info["workspace_bytes"] <= B.OPTCC_STATIC_WORKSPACE_BYTES
    assert lib.optcc_execute_shard(small.handle, fake, C.c_void_p(0x100), None, 2, 2) == B.OPTCC_EINVAL
    assert lib.optcc_execute_shard(small.handle, fake, C.c_void_p(0x100), None, 0, 0) == B.OPTCC_EINVAL
    out = B.optcc_verify_result_t()
    assert lib.optcc_verify_shard(small.handle, C.c_void_p(0x100), None, 3, 2, C.byref(out)) == B.OPTCC_EINVAL
    df = B.optcc_plan(p, 1, ell, 4096, W.F32, k=4, exec_mode=B.OPTCC_EXEC_DATAFLOW)
    assert lib.optcc_execute_shard(df.handle, fake, C.c_void_p(0x100), None, 0, 2) == B.OPTCC_EUNSUPPORTED
    assert lib.optcc_verify_shard(df.handle, C.c_void_p(0x100), None, 0, 2, C.byref(out)) == B.OPTCC_EUNSUPPORTED
