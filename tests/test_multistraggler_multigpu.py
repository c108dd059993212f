"""g > 1 with m >= 2 straggler servers -- the case PAPER.md E.5 (:943) leaves without construction, time analysis or
bound -- planned by composing C2's window structure over the leaders with C3's NVLink phases (PLAN_SPEC C3;
SURVEY 8(f)-2).

Pins (the paper prints nothing for this case, so the pins are reductions to its pinned constructions and invariants):
  * with one straggler server the tables are C3's, byte for byte (the library's C3 was pinned before this change);
  * the NIC flows of every leader cycle are exactly C2's flows on q ranks (servers) with that part's sections;
  * exactly-once contributor sets, hazard freedom, Lemma 4 with equality (:340);
  * every single-straggler Theorem-3 bound is a lower bound of the simulated time; the time stays below the composed
    (k + 5.5)-body form and approaches D.3's limit on n/g elements as k grows.
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


def _ell(q, g, sts):
    e = [1.0] * (q * g)
    for v, l in sts.items():
        for i in range(g):
            e[v * g + i] = float(l)
    return e


CASES = [(6, 2, {0: 2.0, 3: 1.5}, 4), (8, 4, {1: 2.0, 2: 2.0, 5: 8.0 / 7.0}, 8), (5, 2, {0: 3.0, 1: 1.25}, 4), (16, 8, {0: 2.0, 7: 4.0 / 3.0}, 8)]


@pytest.mark.parametrize("q,g,sts,k", CASES)
def test_oracle_composed_plan_invariants_and_time(q, g, sts, k):
    p, m = q * g, len(sts)
    n = 4 * g * k * (q - m) * 30
    ell = _ell(q, g, sts)
    plan = OP.build_plan(p, g, ell, n, OP.F32, k=k)
    assert plan.construction == OP.C3 and plan.m == m and plan.H == q - m
    tot = OI.check_plan(plan)
    assert tot["reduce_elems"] == tot["copy_elems"] == (p - 1) * n                  # Lemma 4 with equality
    sim = cost_sim.simulate(plan)
    for l in sts.values():
        assert cf.lb_thm3(p, g, l, n) <= sim["T"]                                    # every one-straggler bound holds
    assert cost_sim.lower_bounds(plan)["table1"] == max(cf.lb_thm3(p, g, l, n) for l in sts.values())
    assert sim["T"] <= cost_sim.paper_closed_form(plan)                              # composed (k + 5.5)-body form
    lim = Fr(n, g) * max(Fr(2 * (q - 1), q - m), Fr(max(sts.values())) + Fr(2 * (m - 1), q - m))
    assert sim["T"] >= lim and float(sim["T"] / lim) <= 1 + 2.5 / k                  # D.3's limit (:831) on n/g elements


@pytest.mark.parametrize("q,g,sts,k", CASES)
def test_nic_flows_of_a_leader_cycle_are_c2_on_the_servers(q, g, sts, k):
    p, m = q * g, len(sts)
    n = 4 * g * k * (q - m) * 30
    plan = OP.build_plan(p, g, _ell(q, g, sts), n, OP.F32, k=k)
    c2 = OP.build_plan(q, 1, [float(sts.get(v, 1.0)) for v in range(q)], n // g, OP.F32, k=k)
    P = plan.H + m - 1
    D = 1 + -(-(g - 2) // P)
    for lam in range(g):
        f = plan.flows[(plan.flows["link"] == OP.NIC) & (plan.flows["part"] == lam)]
        assert (f["src"] % g == lam).all() and (f["dst"] % g == lam).all()           # leaders only (:854)
        got = sorted(zip((f["step"] - D * P).tolist(), (f["src"] // g).tolist(), (f["dst"] // g).tolist(), f["op"].tolist(),
                         f["stage"].tolist(), f["seg"].tolist(), f["sec"].tolist(), (f["off"] - lam * (n // g)).tolist(), f["len"].tolist()))
        want = sorted(zip(c2.flows["step"].tolist(), c2.flows["src"].tolist(), c2.flows["dst"].tolist(), c2.flows["op"].tolist(),
                          c2.flows["stage"].tolist(), c2.flows["seg"].tolist(), c2.flows["sec"].tolist(), c2.flows["off"].tolist(),
                          c2.flows["len"].tolist()))
        assert got == want


def test_one_straggler_server_is_unchanged_c3(golden):
    """m = 1: the generalised step numbering (P = H) must give the tables C3 always had: 186 steps and 243,840 flows
    at config 4 with k = 8, and the <= (k + 5.5) bodies bound of Eq.(21) (:920)."""
    ell = _ell(16, 8, {0: 2.0})
    plan = OP.build_plan(128, 8, ell, 1 << 16, OP.F32, k=8)
    assert plan.n_steps == 186 and len(plan.flows) == 243840
    sim = cost_sim.simulate(plan)
    assert sim["T"] <= cf.T_multigpu_bound(128, 8, 2.0, 8, 1 << 16)


@pytest.mark.parametrize("q,g,sts,k,n,dtype", [(6, 2, {0: 2.0, 3: 1.5}, 4, 30011, 0), (8, 4, {1: 2.0, 2: 2.0, 5: 8.0 / 7.0}, 8, 100003, 1),
                                               (16, 8, {0: 2.0, 7: 4.0 / 3.0}, 0, 1 << 18, 0), (4, 2, {0: 2.0, 1: 1.5}, 4, 9, 0)])
def test_library_equals_oracle(q, g, sts, k, n, dtype):
    p = q * g
    ell = _ell(q, g, sts)
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k)
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k)
    fl, sb, sec, p2p = B.optcc_plan_tables(plan)
    assert fl.tobytes() == oplan.flows.tobytes() and np.array_equal(sb, oplan.step_begin)
    assert np.array_equal(sec, oplan.sec_bounds) and len(p2p) == 0
    assert plan.info["m"] == len(sts) and plan.info["construction"] == OP.C3 and plan.info["k"] == oplan.k
    c = B.optcc_cost(plan)
    sim = cost_sim.simulate(oplan)
    rel = lambda a, b: abs(a - float(b)) <= 1e-12 * abs(float(b))
    assert rel(c["T"], sim["T"]) and rel(c["lb_table1"], cost_sim.lower_bounds(oplan)["table1"])
    assert rel(c["T_closed_form"], cost_sim.paper_closed_form(oplan)) and c["lb_tight"] != c["lb_tight"]
    assert c["lb_table1"] <= c["T"]
    if n >= 1000:                      # (a handful of 16-byte units cannot be split evenly: the form assumes divisibility)
        assert c["T"] <= c["T_closed_form"] * (1 + 1e-3)


@pytest.mark.gpu
@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_PERSISTENT])
@pytest.mark.parametrize("q,g,sts,k,n,dtype", [(6, 2, {0: 2.0, 3: 1.5}, 4, 30011, 0), (8, 4, {1: 2.0, 2: 2.0, 5: 8.0 / 7.0}, 8, 100003, 1)])
def test_gpu_executes_the_composed_plan(q, g, sts, k, n, dtype, exec_mode):
    from paper_2606_01680_b200 import workloads as W
    from paper_2606_01680_b200.device import Session
    p = q * g
    ell = _ell(q, g, sts)
    w = W.Workload("c3m", p, g, tuple(ell), n, dtype, "normal", 1.0, 99)
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=exec_mode)
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k)
    x = W.all_inputs(w)
    s = Session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == 0 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    assert s.verify()["bad_elements"] == 0
    assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()
