"""Ordering (1) of PAPER.md:138 (S1 -> S2 -> S3 -> S4) as a planner option (PLAN_SPEC C1').

Pins for the oracle's construction (paper values / invariants, not its own formula): flow counts per segment
12/12/4/4 at p = 5 (:146); exactly-once contributor sets and hazard freedom; Lemma 4 with equality (:340); the
straggler sends and receives exactly n (l >= 2, Lemma 5 with equality :346) resp. z* n (l < 2, :455) elements;
Theorem 1/6 <= simulated T <= (k+3) bodies; never faster than the canonical ordering-(2) plan, same k -> infinity limit.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import build as optcc_build
from oracle import planner as OP
from oracle import interpreter as OI
from oracle import cost_sim, closed_forms as cf


@pytest.fixture(scope="module", autouse=True)
def _built():
    optcc_build.build()


def _ell(p, r, l):
    e = [1.0] * p
    e[r] = float(l)
    return e


def test_flow_counts_match_the_papers_worked_example():
    """p = 5, l = 2, k = 4 (:146): S1 and S4 each (p-2)(p-1) = 12 flows, S2 and S3 each p-1 = 4 flows per segment."""
    plan = OP.build_plan(5, 1, _ell(5, 0, 2.0), 4 * 4 * 4 * 25, OP.F32, k=4, ordering=1)
    for b in range(4):
        seg = plan.flows[plan.flows["seg"] == b]
        counts = [int((seg["stage"] == st).sum()) for st in (OP.S1, OP.S2, OP.S3, OP.S4)]
        assert counts == [12, 4, 4, 12]
    assert plan.n_steps == (4 + 3) * 4
    assert (plan.flows[plan.flows["stage"] == OP.S2]["op"] == OP.REDUCE).all()      # the straggler adds (:132)
    assert (plan.flows[plan.flows["stage"] == OP.S3]["op"] == OP.COPY).all()


CASES = [(5, 0, 2.0, 4), (5, 2, 1.5, 4), (5, 4, 3.0, 8), (16, 0, 8.0 / 7.0, 8), (4, 1, 2.0, 4), (3, 0, 2.0, 4), (9, 3, 1.25, 12)]


@pytest.mark.parametrize("p,r,l,k", CASES)
def test_oracle_ordering1_invariants_and_time(p, r, l, k):
    n = 4 * (p - 1) * k * 60 * 7
    ell = _ell(p, r, l)
    plan = OP.build_plan(p, 1, ell, n, OP.F32, k=k, ordering=1)
    tot = OI.check_plan(plan)
    assert tot["reduce_elems"] == tot["copy_elems"] == (p - 1) * n                  # Lemma 4 with equality
    sim = cost_sim.simulate(plan)
    vol = n if l >= 2 else cf.zstar_thm6(p, l) * n                                   # :346 / :455
    assert abs(Fr(sim["nic_sent"][r]) - vol) <= 4 * k and abs(Fr(sim["nic_recvd"][r]) - vol) <= 4 * k
    lbs = cost_sim.lower_bounds(plan)
    lim = cf.T_single_limit(p, l, n)
    assert lbs["table1"] <= sim["T"] and lbs["tight"] <= sim["T"]
    assert sim["T"] <= lim * Fr(k + 3, k) == cost_sim.paper_closed_form(plan)
    canon = cost_sim.simulate(OP.build_plan(p, 1, ell, n, OP.F32, k=k))
    assert canon["T"] <= sim["T"]
    assert sim["T"] / lim > 1 and float(sim["T"] / lim) - 1 <= 3.0 / k + 1e-12       # -> the same limit as k grows


def test_ordering1_masks_and_numerics_on_cpu():
    p, n, k = 6, 12345, 4
    ell = _ell(p, 2, 1.5)
    plan = OP.build_plan(p, 1, ell, n, OP.F32, k=k, ordering=1)
    masks, overlaps = OI.element_masks(plan)
    assert overlaps == 0 and (masks == OI.full_mask_words(p)[None, None, :]).all()
    x = np.random.default_rng(3).standard_normal((p, n)).astype(np.float32)
    y = OI.run_f32(plan, x)
    assert (y == y[0]).all()
    assert np.allclose(y[0], x.astype(np.float64).sum(0), rtol=0, atol=p * 2.0 ** -23 * np.abs(x).sum(0).max())


@pytest.mark.parametrize("p,r,l,k,n,dtype", [(5, 0, 2.0, 4, 4803, 0), (5, 2, 1.5, 4, 50003, 1), (16, 9, 8.0 / 7.0, 8, 123457, 0),
                                             (3, 0, 2.0, 4, 7, 0), (32, 31, 3.0, 12, 999983, 1), (32, 0, 2.0 - 1.0 / 31.0, 0, 1 << 20, 0)])
def test_library_ordering1_equals_oracle(p, r, l, k, n, dtype):
    ell = _ell(p, r, l)
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, ordering=1)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k, ordering=1)
    fl, sb, sec, p2p = B.optcc_plan_tables(plan)
    assert fl.tobytes() == oplan.flows.tobytes() and np.array_equal(sb, oplan.step_begin)
    assert np.array_equal(sec, oplan.sec_bounds) and np.array_equal(p2p, oplan.p2p_bounds)
    assert plan.info["k"] == oplan.k and plan.info["n_steps"] == (oplan.k + 3) * (p - 1)
    c = B.optcc_cost(plan)
    sim = cost_sim.simulate(oplan)
    assert abs(c["T"] - float(sim["T"])) <= 1e-12 * c["T"]
    assert abs(c["T_closed_form"] - float(cost_sim.paper_closed_form(oplan))) <= 1e-12 * c["T_closed_form"]


def test_ordering1_errors():
    for kw, code in ((dict(p=7, ell=[2.0, 1.5] + [1.0] * 5), "EUNSUPPORTED"), (dict(p=6, ell=[1.0] * 6), "EUNSUPPORTED")):
        with pytest.raises(OP.PlanError) as eo:
            OP.build_plan(kw["p"], 1, kw["ell"], 1000, OP.F32, ordering=1)
        assert eo.value.code == code
        with pytest.raises(B.OptccError) as el:
            B.optcc_plan(kw["p"], 1, kw["ell"], 1000, B.OPTCC_F32, ordering=1)
        assert el.value.name == code
    with pytest.raises(B.OptccError) as el:
        B.optcc_plan(5, 1, _ell(5, 0, 2.0), 1000, B.OPTCC_F32, ordering=4)
    assert el.value.name == "EINVAL"
    with pytest.raises(OP.PlanError):
        OP.build_plan(5, 1, _ell(5, 0, 2.0), 1000, OP.F32, ordering=4)
    assert B.optcc_plan_tables(B.optcc_plan(5, 1, _ell(5, 0, 2.0), 1000, B.OPTCC_F32, ordering=2))[0].tobytes() == \
        B.optcc_plan_tables(B.optcc_plan(5, 1, _ell(5, 0, 2.0), 1000, B.OPTCC_F32))[0].tobytes()


@pytest.mark.gpu
@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_PERSISTENT, B.OPTCC_EXEC_PER_STEP])
@pytest.mark.parametrize("p,r,l,k,n,dtype", [(5, 2, 1.5, 4, 50003, 1), (16, 0, 8.0 / 7.0, 8, 2 ** 17 + 3, 0), (4, 0, 2.0, 4, 100003, 0)])
def test_gpu_executes_ordering1(p, r, l, k, n, dtype, exec_mode):
    from paper_2606_01680_b200 import workloads as W
    from paper_2606_01680_b200.device import Session
    ell = _ell(p, r, l)
    w = W.Workload("ord1", p, 1, tuple(ell), n, dtype, "normal", 1.0, 55)
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, ordering=1, exec_mode=exec_mode)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k, ordering=1)
    x = W.all_inputs(w)
    s = Session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == 0 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    assert s.verify()["bad_elements"] == 0
    assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()
