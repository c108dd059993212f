"""Pins for oracle/planner.py + interpreter.py + cost_sim.py: worked example p=5,
Eq.(1)/(2) as equalities of rationals, exactly-once masks, Lemma 4/5 volumes, bounds of App. D/E."""
from fractions import Fraction as Fr

import numpy as np
import pytest

from oracle import closed_forms as cf
from oracle import cost_sim, interpreter
from oracle import planner as P


def ell_vec(p, d):
    return [float(d.get(i, 1.0)) for i in range(p)]


def count(plan, **kw):
    m = np.ones(len(plan.flows), dtype=bool)
    for key, v in kw.items():
        m &= plan.flows[key] == v
    return int(m.sum())


def test_worked_example_p5_l2_flow_counts(golden):
    # :146 GPU 0 straggler, 50 % throughput; 12/12/4/4 flows per segment; k=4 -> 5 bodies (:163, :169)
    k = 4
    plan = P.build_plan(5, 1, ell_vec(5, {0: 2.0}), 4 * k * 4 * 25, P.F32, k=k)
    interpreter.check_plan(plan)
    for b in range(k):
        assert count(plan, stage=P.S1, seg=b) == golden["p5_l2_S1_flows_per_segment"]
        assert count(plan, stage=P.S4, seg=b) == golden["p5_l2_S4_flows_per_segment"]
        assert count(plan, stage=P.S2, seg=b) == golden["p5_l2_S2_flows_per_segment"]
        assert count(plan, stage=P.S3, seg=b) == golden["p5_l2_S3_flows_per_segment"]
    assert count(plan, stage=P.BUB_UP) == 0 and count(plan, stage=P.BUB_DOWN) == 0   # l=2: no bubbles (:163)
    H = 4
    assert plan.n_steps == golden["p5_k4_parallel_bodies"] * H
    # every stage of one segment fits in 2(p-1) = 8 unit slots: S1 is 3 hops, S2/S3 4 flows of 2 slots
    assert (5 - 2) <= golden["p5_l2_slots_per_stage"] and 4 * 2 == golden["p5_l2_slots_per_stage"]
    # all S1/S4 flows are healthy<->healthy, all S2/S3 flows touch the straggler (:142 disjoint links)
    f = plan.flows
    ring = (f["stage"] == P.S1) | (f["stage"] == P.S4)
    assert ((f["src"][ring] != 0) & (f["dst"][ring] != 0)).all()
    assert (f["dst"][f["stage"] == P.S2] == 0).all() and (f["src"][f["stage"] == P.S3] == 0).all()


@pytest.mark.parametrize("p", [3, 4, 5, 16])
@pytest.mark.parametrize("ell", [2.0, 3.0, 2.5])
@pytest.mark.parametrize("k", [4, 8, 20])
def test_eq1_exact(p, ell, k):
    n = 4 * k * (p - 1) * 3
    plan = P.build_plan(p, 1, ell_vec(p, {0: ell}), n, P.F32, k=k)
    interpreter.check_plan(plan)
    sim = cost_sim.simulate(plan)
    assert sim["T"] == cf.T_eq1(p, ell, k, n)                      # Eq.(1) :173, equality of rationals
    assert sim["nic_sent"][0] == n and sim["nic_recvd"][0] == n     # Lemma 5 with equality (:344)


# (p, ell as exact binary-friendly rational, U multiplier) with (2-l)/((p-2)l+2) = a/b exactly representable
@pytest.mark.parametrize("p,ell,den", [(5, 1.5, 13), (3, 1.5, 7), (4, 1.5, 10), (5, 1.25, 23), (16, 1.5, 46), (6, 1.0 + 2.0 ** -3, 52)])
@pytest.mark.parametrize("k", [4, 8, 20])
def test_eq2_exact(p, ell, den, k):
    l = Fr(ell)
    frac = (2 - l) / ((p - 2) * l + 2)
    assert frac.denominator == den or den % frac.denominator == 0
    U = den * k * (p - 1) * 2
    n = 4 * U
    plan = P.build_plan(p, 1, ell_vec(p, {0: ell}), n, P.F32, k=k)
    assert Fr(plan.U_p2p, plan.U) == frac                           # a2: P2P share (:746-748)
    interpreter.check_plan(plan)
    sim = cost_sim.simulate(plan)
    assert sim["T"] == cf.T_eq2(p, ell, k, n)                       # Eq.(2) :185/:752, equality of rationals
    # Theorem 6 optimum: straggler sends and receives exactly z* n (:455)
    assert sim["nic_sent"][0] == cf.zstar_thm6(p, ell) * n
    assert sim["nic_recvd"][0] == cf.zstar_thm6(p, ell) * n
    # section size s' (:748) and P2P piece (2-l)s'/l (:744)
    s = cf.section_size_bubble(p, k, ell, n)
    f = plan.flows
    assert set(f["len"][f["stage"] == P.S1].tolist()) == {int(s)} and s.denominator == 1
    assert set(f["len"][f["stage"] == P.BUB_UP].tolist()) == {int(cf.p2p_per_segment(p, k, ell, n))}


def test_straggler_position_does_not_matter():
    for sg in range(5):
        n = 4 * 13 * 4 * 4
        plan = P.build_plan(5, 1, ell_vec(5, {sg: 1.5}), n, P.F32, k=4)
        interpreter.check_plan(plan)
        assert cost_sim.simulate(plan)["T"] == cf.T_eq2(5, 1.5, 4, n)


@pytest.mark.parametrize("p", [3, 4, 6, 16, 33])
def test_c0_plain_ring_hits_T0(p):
    n = 4 * p * 5
    plan = P.build_plan(p, 1, [1.0] * p, n, P.F32)
    assert plan.construction == P.C0 and plan.k == 1 and plan.n_steps == 2 * (p - 1)
    interpreter.check_plan(plan)
    sim = cost_sim.simulate(plan)
    assert sim["T"] == sim["T0"] == 2 * (p - 1) * Fr(n, p)          # :72 attained by Ring AllReduce
    assert len(plan.flows) == 2 * p * (p - 1)


@pytest.mark.parametrize("p,ells", [(7, {0: 2.0, 1: 4.0 / 3.0}), (7, {0: 1.5, 1: 1.5}), (9, {2: 3.0, 5: 2.0, 7: 1.25}),
                                    (16, {3: 8.0 / 7.0, 9: 4.0 / 3.0}), (6, {0: 2.0, 1: 2.0, 2: 2.0})])
@pytest.mark.parametrize("k", [4, 8])
def test_c2_multi_straggler(p, ells, k):
    m = len(ells)
    H = p - m
    n = 4 * k * H * 6
    plan = P.build_plan(p, 1, ell_vec(p, ells), n, P.F32, k=k)
    assert plan.construction == P.C2 and plan.H == H and plan.n_steps == (k + 1) * (p - 1)   # :788 p-1 windows
    interpreter.check_plan(plan)
    sim = cost_sim.simulate(plan)
    lv = sorted(ells.values(), reverse=True)
    assert [plan.ell[s] for s in plan.stragglers] == lv              # :78 order
    assert cf.lb_thm2(p, lv, n) <= sim["T"] <= cf.T_multi_paper(p, lv, k, n)     # Thm 2 <= T <= (k+4) T_body (:809)
    # per segment each straggler exchanges one flow with every healthy GPU in each direction (:773-774)
    for sg in ells:
        assert count(plan, stage=P.S2, dst=sg, seg=0) == H and count(plan, stage=P.S3, src=sg, seg=0) == H
        assert sim["nic_sent"][sg] == n and sim["nic_recvd"][sg] == n            # Lemma 8 with equality
    assert set(plan.flows["len"].tolist()) == {n // (k * H)}                     # s = n/(k(p-m)) :770


def test_c2_window_structure():
    # :788 "p-m-1 windows carry merged ring flows and m windows carry straggler communication" -- per healthy GPU
    p, k = 7, 4
    plan = P.build_plan(p, 1, ell_vec(p, {0: 2.0, 1: 4.0 / 3.0}), 4 * k * 5 * 3, P.F32, k=k)
    f = plan.flows
    body1 = f[(f["step"] >= 6) & (f["step"] < 12)]
    for hr in range(2, 7):
        sends = body1[body1["src"] == hr]
        ring_w = set((sends["step"][(sends["stage"] == P.S1)] - 6).tolist())
        str_w = set((sends["step"][(sends["stage"] == P.S2)] - 6).tolist())
        assert len(ring_w) == p - 2 - 1 and len(str_w) == 2 and not (ring_w & str_w)


@pytest.mark.parametrize("g,q,ell", [(2, 4, 2.0), (4, 5, 2.0), (4, 4, 1.5), (8, 3, 3.0), (2, 3, 8.0 / 7.0)])
@pytest.mark.parametrize("k", [8, 24])
def test_c3_multi_gpu(g, q, ell, k):
    p = g * q
    H = q - 1
    n = 4 * g * k * H * 2
    for sv in (0, q - 1):
        ells = ell_vec(p, {sv * g + i: ell for i in range(g)})
        plan = P.build_plan(p, g, ells, n, P.F32, k=k)
        assert plan.construction == P.C3
        interpreter.check_plan(plan)
        sim = cost_sim.simulate(plan)
        assert cf.lb_thm13(p, g, ell, n) <= sim["T"] <= cf.T_multigpu_bound(p, g, ell, k, n)   # Thm 13 <= T <= Eq.(21)/(22)
        assert set(plan.flows["len"].tolist()) == {n // (g * k * H)}             # s = n/(gk(q-1)) :843
        f = plan.flows
        nic = f[f["link"] == P.NIC]
        # leaders only: a NIC flow joins local GPU lambda of two servers (:854)
        assert ((nic["src"] % g) == nic["part"]).all() and ((nic["dst"] % g) == nic["part"]).all()
        nv = f[f["link"] == P.NVLINK]
        assert ((nv["src"] // g) == (nv["dst"] // g)).all()
        col = nv[nv["stage"] == P.N_COLLECT]
        dis = nv[nv["stage"] == P.N_DISTRIBUTE]
        assert (((col["src"] % g) - (col["dst"] % g)) % g == 1).all()            # backward ring (:894)
        assert (((dis["dst"] % g) - (dis["src"] % g)) % g == 1).all()            # forward ring
        assert ((col["src"] % g) != col["part"]).all()                           # leader only receives
        assert ((dis["dst"] % g) != dis["part"]).all()                           # leader sends first, never receives
        # Lemma 11/12 with equality: inter-server traffic 2(q-1)n, straggler server n each way
        assert int(nic["len"].sum()) == 2 * (q - 1) * n
        srv = lambda r: r // g
        assert int(nic["len"][srv(nic["src"]) == sv].sum()) == n and int(nic["len"][srv(nic["dst"]) == sv].sum()) == n


def test_validation_errors():
    with pytest.raises(P.PlanError) as e:
        P.build_plan(2, 1, [1, 2], 100, P.F32)
    assert e.value.code == "EINVAL"                                  # p >= 3 (:68)
    for bad in ([0.5, 1, 1, 1], [float("nan"), 1, 1, 1], [float("inf"), 1, 1, 1]):
        with pytest.raises(P.PlanError):
            P.build_plan(4, 1, bad, 100, P.F32)
    with pytest.raises(P.PlanError) as e:
        P.build_plan(4, 1, [2, 2, 2, 1], 100, P.F32)
    assert e.value.code == "EINVAL"                                  # < 2 healthy
    with pytest.raises(P.PlanError) as e:
        P.build_plan(8, 2, [2, 1, 1, 1, 1, 1, 1, 1], 100, P.F32)
    assert e.value.code == "EINVAL"                                  # mixed ell in a server (:274)
    with pytest.raises(P.PlanError) as e:
        P.build_plan(8, 2, [1] * 8, 100, P.F32)
    assert e.value.code == "EUNSUPPORTED"                            # g > 1 without a straggler: NCCL's own ring (:88)
    assert P.build_plan(8, 2, [2, 2, 1.5, 1.5, 1, 1, 1, 1], 100, P.F32).construction == P.C3   # E.5 :943: composed plan
    with pytest.raises(P.PlanError):
        P.build_plan(4, 1, [2, 1, 1, 1], 100, P.F32, k=6)            # k multiple of 4 (:155)
    with pytest.raises(P.PlanError):
        P.build_plan(4, 1, [2, 1, 1, 1], 0, P.F32)
    with pytest.raises(P.PlanError):
        P.build_plan(6, 4, [1] * 6, 10, P.F32)


@pytest.mark.parametrize("n", [1, 3, 5, 17, 63, 1001, 4099])
@pytest.mark.parametrize("cfg", [(4, 1, {0: 2.0}), (5, 1, {2: 1.5}), (7, 1, {0: 2.0, 3: 1.25}), (6, 2, {0: 2.0, 1: 2.0}), (5, 1, {})])
@pytest.mark.parametrize("dtype", [P.F32, P.BF16])
def test_ragged_and_tiny_n_stay_exactly_once(n, cfg, dtype):
    p, g, ells = cfg
    plan = P.build_plan(p, g, ell_vec(p, ells), n, dtype, k=4)
    interpreter.check_plan(plan)       # zero-length flows dropped, everything still covered exactly once
    A = plan.A
    f = plan.flows
    assert (f["off"] % A == 0).all()                                  # R3: 16-byte aligned starts
    ragged = f["len"] % A != 0
    assert ((f["off"] + f["len"])[ragged] == n).all()                 # only a region ending at n may be ragged


def test_element_masks_agree_with_set_walk():
    for p, g, ells, n in [(5, 1, {0: 1.5}, 203), (6, 2, {4: 2.0, 5: 2.0}, 97), (7, 1, {1: 2.0, 2: 3.0}, 50)]:
        plan = P.build_plan(p, g, ell_vec(p, ells), n, P.F32, k=4)
        masks, overlaps = interpreter.element_masks(plan)
        assert overlaps == 0
        assert (masks == interpreter.full_mask_words(p)[None, None, :]).all()


def test_check_plan_catches_mistakes():
    plan = P.build_plan(5, 1, ell_vec(5, {0: 1.5}), 4 * 13 * 16, P.F32, k=4)
    # dropped flow -> someone misses a contributor
    bad = P.build_plan(5, 1, ell_vec(5, {0: 1.5}), 4 * 13 * 16, P.F32, k=4)
    bad.flows = np.delete(bad.flows, 7)
    bad.step_begin = np.searchsorted(bad.flows["step"], np.arange(bad.n_steps + 1)).astype(np.uint32)
    with pytest.raises(interpreter.PlanViolation):
        interpreter.check_plan(bad)
    # duplicated reduce -> overlapping contributor sets
    bad = P.build_plan(5, 1, ell_vec(5, {0: 1.5}), 4 * 13 * 16, P.F32, k=4)
    i = int(np.nonzero(bad.flows["stage"] == P.S3)[0][0])
    dup = bad.flows[i:i + 1].copy()
    dup["step"] += 4
    bad.flows = np.sort(np.concatenate([bad.flows, dup]), order=["step", "link", "stage", "src", "dst", "off"])
    bad.step_begin = np.searchsorted(bad.flows["step"], np.arange(bad.n_steps + 1)).astype(np.uint32)
    with pytest.raises(interpreter.PlanViolation):
        interpreter.check_plan(bad)
    # swapped src/dst of a copy -> wrong data direction
    bad = P.build_plan(5, 1, ell_vec(5, {0: 1.5}), 4 * 13 * 16, P.F32, k=4)
    i = int(np.nonzero(bad.flows["stage"] == P.S2)[0][0])
    bad.flows["src"][i], bad.flows["dst"][i] = bad.flows["dst"][i], bad.flows["src"][i]
    with pytest.raises(interpreter.PlanViolation):
        interpreter.check_plan(bad)
    interpreter.check_plan(plan)


def test_auto_k_rule():
    # PLAN_SPEC §2 'k': finite-k factor <= 1.05, section >= 64 KiB, multiple of 4, >= 4
    mk = lambda p, g, e, n, dt: P.build_plan(p, g, e, n, dt, k=0).k
    assert mk(4, 1, ell_vec(4, {0: 2.0}), 2 ** 20, P.F32) == 20
    assert mk(16, 1, ell_vec(16, {0: 8 / 7}), 2 ** 26, P.F32) == 4
    assert mk(32, 1, ell_vec(32, {0: 1.6}), 2 ** 25, P.F32) == 12
    assert mk(32, 1, ell_vec(32, {0: 3.0}), 2 ** 25, P.F32) == 20
    assert mk(64, 1, ell_vec(64, {5: 8 / 7, 17: 4 / 3, 40: 2.0}), 2 ** 24, P.BF16) == 8      # capped by 64 KiB sections
    assert mk(128, 8, ell_vec(128, {r: 2.0 for r in range(8)}), 2 ** 22, P.F32) == 4
    assert mk(4, 1, ell_vec(4, {0: 2.0}), 100, P.F32) == 4


def test_planner_is_fast_at_p1024():
    # :189 "For p=1024 ... generated in under 1 ms on a single CPU core" is the C++ planner's target; the
    # pure-Python oracle only has to stay usable.
    import time
    t = time.time()
    plan = P.build_plan(1024, 1, ell_vec(1024, {0: 2.0}), 2 ** 24, P.F32, k=4)
    assert time.time() - t < 120 and len(plan.flows) == 4 * (2 * 1022 * 1023 + 2 * 1023)
