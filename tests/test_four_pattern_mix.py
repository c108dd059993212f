"""The four-pattern mix of PAPER.md:144-155 as a planner option (ordering = 3, PLAN_SPEC C1'').

Figures 5-6 (the slot-exact layout) are absent from PAPER.md; the construction keeps what the text fixes, and these
tests pin exactly that: patterns A, C use ordering (1) and B, D ordering (2) (:148-151); k/4 segments per pattern
(:155); 12/12/4/4 flows per segment at p = 5 (:146); k+1 parallel bodies, the head and the tail partly filled and every
other body holding one part of each of the four patterns (:169); no NIC carries two flows at once (:124, the port
model); at l = 2 no port idles in the steady state ("the body has no idle bubbles", :163); completion time = Eq.(1)
(:173) at l = 2 and Eq.(2) (:185) for l < 2 as EQUALITIES of rationals for divisible n, and between the lower bound
and Eq.(1) for l > 2; exactly-once contributor sets, hazard freedom, Lemma 4 / 5 with equality, z* n straggler volume.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import build as optcc_build
from paper_2606_01680_b200 import workloads as W
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


def test_patterns_stages_and_bodies_of_the_worked_example(golden):
    """p = 5, l = 2, k = 4 (:146, Fig. 6 caption :163): 12/12/4/4 flows per segment, 5 parallel bodies."""
    p, k = 5, 4
    H = p - 1
    plan = OP.build_plan(p, 1, _ell(p, 0, 2.0), 4 * H * k * 25, OP.F32, k=k, ordering=3)
    assert plan.n_steps == int(golden["p5_k4_parallel_bodies"]) * H == (k + 1) * H
    fl = plan.flows
    for b in range(k):
        seg = fl[fl["seg"] == b]
        assert [int((seg["stage"] == st).sum()) for st in (OP.S1, OP.S2, OP.S3, OP.S4)] == \
            [int(golden["p5_l2_S%d_flows_per_segment" % i]) for i in (1, 2, 3, 4)]
        body_of = {st: set((seg["step"][seg["stage"] == st] // H).tolist()) for st in (OP.S1, OP.S2, OP.S3, OP.S4)}
        assert all(len(v) == 1 for v in body_of.values())             # one stage per body: 2(p-1) slots per stage (:146)
        order = sorted((min(v), st) for st, v in body_of.items())
        seq = [st for _, st in order]
        if b % 4 in (0, 2):      # patterns A, C: S1 -> S2 -> S3 -> S4, the straggler performs the last add (:148, :150)
            assert seq == [OP.S1, OP.S2, OP.S3, OP.S4]
            assert (seg["op"][seg["stage"] == OP.S2] == OP.REDUCE).all() and (seg["op"][seg["stage"] == OP.S3] == OP.COPY).all()
        else:                    # patterns B, D: S3 -> S1 -> S4 -> S2, the straggler uploads its raw data first (:149, :151)
            assert seq == [OP.S3, OP.S1, OP.S4, OP.S2]
            assert (seg["op"][seg["stage"] == OP.S3] == OP.REDUCE).all() and (seg["op"][seg["stage"] == OP.S2] == OP.COPY).all()
        assert [bd - order[0][0] for bd, _ in order] == [0, 1, 2, 3]   # four consecutive bodies per pattern ...
        assert 4 * 2 * H == int(golden["p5_l2_slots_per_pattern"]) and 2 * H == int(golden["p5_l2_slots_per_stage"])   # ... of 8 slots (:146)


@pytest.mark.parametrize("p,k", [(5, 4), (5, 8), (4, 12), (9, 20)])
def test_every_full_body_holds_one_part_of_each_pattern(p, k):
    """:169 "k-1 steady-state bodies that each contain one part from each of the four patterns, plus one startup body
    at the head and one drain body at the tail"."""
    H = p - 1
    plan = OP.build_plan(p, 1, _ell(p, 1, 2.0), 4 * H * k * 6, OP.F32, k=k, ordering=3)
    fl = plan.flows
    body = fl["step"] // H
    for beta in range(k + 1):
        inst = {(int(s) % 4, int(st)) for s, st in zip(fl["seg"][body == beta], fl["stage"][body == beta])}
        pats = sorted(pt for pt, _ in inst)
        if beta == 0:
            assert pats == [0, 1]                      # head: the first stages of A and B
        elif beta == k:
            assert pats == [2, 3]                      # tail: the last stages of C and D
        else:
            assert pats == [0, 1, 2, 3] and len(inst) == 4


@pytest.mark.parametrize("p,ell,den", [(5, 1.5, 13), (3, 1.5, 7), (4, 1.5, 10), (5, 1.25, 23), (16, 1.5, 46), (6, 1.0 + 2.0 ** -3, 52)])
@pytest.mark.parametrize("k", [4, 8, 20])
def test_mix_reaches_eq2_exactly(p, ell, den, k):
    """l < 2 with bubble filling: the simulated completion time of the mix equals Eq.(2) (:185, :752) as a rational."""
    n = 4 * den * k * (p - 1) * 2
    plan = OP.build_plan(p, 1, _ell(p, 0, ell), n, OP.F32, k=k, ordering=3)
    OI.check_plan(plan)
    sim = cost_sim.simulate(plan)
    assert sim["T"] == cf.T_eq2(p, ell, k, n)
    assert sim["nic_sent"][0] == sim["nic_recvd"][0] == cf.zstar_thm6(p, ell) * n       # Theorem 6 optimum (:455)


@pytest.mark.parametrize("p", [3, 4, 5, 8, 16])
@pytest.mark.parametrize("k", [4, 8, 20])
def test_mix_at_ell_2_has_no_idle_port_in_the_steady_state(p, k):
    """l = 2 (:163, :175): T = Eq.(1) exactly, and every NIC port of every rank is busy for k of the k+1 bodies -- the
    head and tail bodies are the only idle time ("the body has no idle bubbles")."""
    n = 4 * (p - 1) * k * 6
    plan = OP.build_plan(p, 1, _ell(p, 0, 2.0), n, OP.F32, k=k, ordering=3)
    OI.check_plan(plan)
    sim = cost_sim.simulate(plan)
    assert sim["T"] == cf.T_eq1(p, 2.0, k, n) == Fr(2 * n * (k + 1), k)
    for r in range(p):
        assert sim["load_send"][r] == sim["load_recv"][r] == sim["T"] * Fr(k, k + 1)
    assert sim["nic_sent"][0] == sim["nic_recvd"][0] == n                               # Lemma 5 with equality (:346)


@pytest.mark.parametrize("p,r,l,k", [(5, 0, 3.0, 8), (16, 4, 2.5, 12), (4, 3, 8.0, 4), (9, 2, 2.25, 20)])
def test_mix_straggler_bound_regime(p, r, l, k):
    """l > 2: on or above both lower bounds, never slower than Eq.(1)'s k+1 straggler-bound bodies (the event
    simulation lets the last Stage-2 flows start before their body), same k -> infinity limit."""
    n = 4 * (p - 1) * k * 6
    plan = OP.build_plan(p, 1, _ell(p, r, l), n, OP.F32, k=k, ordering=3)
    tot = OI.check_plan(plan)
    assert tot["reduce_elems"] == tot["copy_elems"] == (p - 1) * n                      # Lemma 4 with equality (:340)
    sim = cost_sim.simulate(plan)
    lbs = cost_sim.lower_bounds(plan)
    assert lbs["table1"] <= sim["T"] and lbs["tight"] <= sim["T"] <= cf.T_eq1(p, l, k, n)
    assert sim["T"] >= cf.T_single_limit(p, l, n)


def test_mix_masks_and_numerics_on_cpu():
    p, n, k = 6, 12345, 8
    ell = _ell(p, 2, 1.5)
    plan = OP.build_plan(p, 1, ell, n, OP.F32, k=k, ordering=3)
    masks, overlaps = OI.element_masks(plan)
    assert overlaps == 0 and (masks == OI.full_mask_words(p)[None, None, :]).all()
    x = np.random.default_rng(3).standard_normal((p, n)).astype(np.float32)
    y = OI.run_f32(plan, x)
    assert (y == y[0]).all()
    assert np.allclose(y[0], x.astype(np.float64).sum(0), rtol=0, atol=p * 2.0 ** -23 * np.abs(x).sum(0).max())


LIB_CASES = [(5, 0, 2.0, 4, 4803, 0), (5, 2, 1.5, 4, 50003, 1), (16, 9, 8.0 / 7.0, 8, 123457, 0), (3, 0, 2.0, 4, 7, 0),
             (32, 31, 3.0, 12, 999983, 1), (32, 0, 2.0 - 1.0 / 31.0, 0, 1 << 20, 0), (9, 4, 1.25, 20, 77777, 0)]


@pytest.mark.parametrize("p,r,l,k,n,dtype", LIB_CASES)
def test_library_mix_equals_oracle(p, r, l, k, n, dtype):
    ell = _ell(p, r, l)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k, ordering=3)
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, ordering=3)
    fl, sb, sec, p2p = B.optcc_plan_tables(plan)
    assert fl.tobytes() == oplan.flows.tobytes() and np.array_equal(sb, oplan.step_begin)
    assert np.array_equal(sec, oplan.sec_bounds) and np.array_equal(p2p, oplan.p2p_bounds)
    c = B.optcc_cost(plan)
    sim = cost_sim.simulate(oplan)
    assert abs(c["T"] - float(sim["T"])) <= 1e-12 * float(sim["T"])
    assert abs(c["T_closed_form"] - float(cost_sim.paper_closed_form(oplan))) <= 1e-12 * c["T_closed_form"]


def test_mix_errors():
    for kw in (dict(p=7, g=1, ell=[2.0, 1.5] + [1.0] * 5), dict(p=6, g=1, ell=[1.0] * 6), dict(p=8, g=2, ell=[2.0, 2.0] + [1.0] * 6)):
        with pytest.raises(OP.PlanError) as eo:
            OP.build_plan(kw["p"], kw["g"], kw["ell"], 1000, OP.F32, ordering=3)
        assert eo.value.code == "EUNSUPPORTED"
        with pytest.raises(B.OptccError) as el:
            B.optcc_plan(kw["p"], kw["g"], kw["ell"], 1000, B.OPTCC_F32, ordering=3)
        assert el.value.name == "EUNSUPPORTED"


@pytest.mark.gpu
@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_COLUMN, B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_PERSISTENT, B.OPTCC_EXEC_PER_STEP])
@pytest.mark.parametrize("p,r,l,k,n,dtype", [(5, 2, 1.5, 4, 50003, 1), (16, 0, 8.0 / 7.0, 8, 2 ** 17 + 3, 0), (4, 0, 2.0, 4, 100003, 0),
                                             (9, 4, 3.0, 12, 400001, 0)])
def test_gpu_executes_the_mix(p, r, l, k, n, dtype, exec_mode):
    from paper_2606_01680_b200.device import Session
    ell = _ell(p, r, l)
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, exec_mode=exec_mode, ordering=3)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k, ordering=3)
    x = W.all_inputs(W.Workload("mix", p, 1, tuple(ell), n, dtype, "normal", 1.0, 77))
    s = Session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0
    assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()
