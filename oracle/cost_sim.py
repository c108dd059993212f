"""Port-model event simulation of a plan in exact rationals (PLAN_SPEC §6).

Test infrastructure only (see oracle/__init__.py).  Model: PAPER.md:68 (healthy NIC one element per
time unit, slowdown l -> l time units per element), :124 (a NIC handles one incoming flow at a time),
:134 (full duplex: one send and one receive), :356/:432 (a transfer incident to a straggler costs l),
:847-848/:908 (NVLink lane at (g-1) x NIC speed, per GPU and direction).
"""
from fractions import Fraction as Fr

from . import planner as P
from . import closed_forms as cf


def simulate(plan, alpha=0, beta=1, alpha_latency=0, sync=0):
    """Returns dict(T, T0, ratio, port loads ...) with Fractions.  Flows are processed in table order.

    alpha occupies the ports (a fixed cost per flow on its send and receive port).  alpha_latency and sync are the
    latency-type fixed costs of PLAN_SPEC 6 (PAPER.md:201 fn.5: about 14 % of the fault-free ring's time is fixed
    overhead; :199, :217: inter-GPU dependencies are enforced with P2P sync messages): the ports are busy for the
    transfer only, the data is usable alpha_latency after the transfer ends, and a flow that has to wait for data
    (rather than for a port) learns about it `sync` later."""
    p, g = plan.p, plan.g
    ell = [Fr(x) for x in plan.ell]
    alpha, beta, alat, sync = Fr(alpha), Fr(beta), Fr(alpha_latency), Fr(sync)
    send = {}   # (rank, link) -> free time
    recv = {}
    wfin, rfin = {}, {}
    zero = Fr(0)
    T = zero
    load_send = [zero] * p   # NIC busy time per rank (for the fluid bound of brute_force)
    load_recv = [zero] * p
    nic_sent = [0] * p       # NIC elements sent / received per rank (Lemma 5 / :455)
    nic_recvd = [0] * p
    for f in plan.flows:
        s, d, off, ln, link = int(f["src"]), int(f["dst"]), int(f["off"]), int(f["len"]), int(f["link"])
        if link == P.NIC:
            dur = alpha + beta * ln * max(ell[s], ell[d])
        else:
            dur = alpha + beta * Fr(ln, g - 1)
        dep = max(wfin.get((s, off), zero), wfin.get((d, off), zero), rfin.get((d, off), zero))
        start = max(send.get((s, link), zero), recv.get((d, link), zero), dep + sync if dep > zero else zero)
        fin = start + dur
        send[(s, link)] = fin
        recv[(d, link)] = fin
        rfin[(s, off)] = max(rfin.get((s, off), zero), fin)   # the source range may be overwritten once it has been sent
        wfin[(d, off)] = fin + alat                            # the data is usable alpha_latency after the transfer
        if fin + alat > T:
            T = fin + alat
        if link == P.NIC:
            load_send[s] += dur
            load_recv[d] += dur
            nic_sent[s] += ln
            nic_recvd[d] += ln
    t0 = cf.T0(p, plan.n, g)
    return {"T": T, "T0": t0, "ratio": T / t0, "load_send": load_send, "load_recv": load_recv,
            "nic_sent": nic_sent, "nic_recvd": nic_recvd,
            "fluid": max(max(load_send), max(load_recv))}


def lower_bounds(plan):
    """Table-1 bound (Thm 1/2/3) and tight bound (Thm 6/13; None for m > 1, Remark 9 :519) for a plan."""
    p, g, n = plan.p, plan.g, plan.n
    ells = [plan.ell[v * g] for v in plan.stragglers]
    if plan.m == 0:
        t0 = cf.T0(p, n, g)
        return {"table1": t0, "tight": t0}
    if g > 1 and plan.m > 1:
        # E.5 (:943) gives no bound for several straggler servers; every single-straggler bound stays valid (making the
        # other stragglers healthy cannot slow the AllReduce down), so the largest Theorem-3 value is a lower bound
        return {"table1": max(cf.lb_thm3(p, g, l, n) for l in ells), "tight": None}
    if g > 1:
        return {"table1": cf.lb_thm3(p, g, ells[0], n), "tight": cf.lb_thm13(p, g, ells[0], n)}
    if plan.m == 1:
        return {"table1": cf.lb_thm1(p, ells[0], n), "tight": cf.lb_thm6(p, ells[0], n)}
    return {"table1": cf.lb_thm2(p, ells, n), "tight": None}


def paper_closed_form(plan):
    """The paper's own finite-k time for the plan's setting: Eq.(1)/(2) (exact for the canonical plan),
    (k+4) T_body (:809) and Eq.(21)/(22) (:920-926) as upper bounds."""
    p, g, n, k = plan.p, plan.g, plan.n, plan.k
    ells = [plan.ell[v * g] for v in plan.stragglers]
    if getattr(plan, "schedule", 0) == P.RING_DEGRADED:
        return cf.T_ring_degraded(p, ells, n)
    if plan.m == 0:
        return cf.T0(p, n, g)
    if g > 1 and plan.m > 1:
        return cf.T_multigpu_multi_composed(p, g, ells, k, n)
    if g > 1:
        return cf.T_multigpu_bound(p, g, ells[0], k, n)
    if plan.m == 1 and getattr(plan, "ordering", 2) == 1:
        return cf.T_single_limit(p, ells[0], n) * cf.Fr(k + 3, k)    # one stage per body: k + 3 bodies (PLAN_SPEC C1')
    if plan.m == 1:
        return cf.T_single(p, ells[0], k, n)
    return cf.T_multi_paper(p, ells, k, n)
