"""Randomised CPU cross-check of the two independent planners and cost models (no GPU): for seeded random
(p, g, ell, n, dtype, k, ordering / schedule) the C++ tables equal the oracle's byte for byte, the oracle's invariants
hold (exactly-once, hazards, Lemma 4), and optcc_cost equals the exact-rational simulation to 1e-12."""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import build as optcc_build
from oracle import planner as OP
from oracle import interpreter as OI
from oracle import cost_sim


@pytest.fixture(scope="module", autouse=True)
def _built():
    optcc_build.build()


ELLS = [8 / 7, 4 / 3, 1.25, 1.5, 1.6, 2.0 - 1.0 / 31.0, 2.0, 2.5, 3.0, 1.0 + 2.0 ** -30]


def _case(rng):
    kind = int(rng.integers(0, 6))
    ordering, schedule = 0, 0
    if kind in (0, 4, 5):
        p, g = int(rng.integers(3, 40)), 1
        st = {int(rng.integers(0, p)): float(rng.choice(ELLS))}
        ordering = 1 if kind == 4 else 0
        schedule = 1 if kind == 5 else 0
    elif kind == 1:
        p, g = int(rng.integers(5, 30)), 1
        m = int(rng.integers(2, min(5, p - 2) + 1))
        st = {int(r): float(rng.choice(ELLS)) for r in rng.choice(p, size=m, replace=False)}
    elif kind == 2:
        g = int(rng.choice([2, 3, 4, 8]))
        q = int(rng.integers(3, 9))
        p = g * q
        m = int(rng.integers(1, min(3, q - 2) + 1))
        st = {}
        for v in rng.choice(q, size=m, replace=False):
            l = float(rng.choice(ELLS))
            for i in range(g):
                st[int(v) * g + i] = l
    else:
        p, g, st = int(rng.integers(3, 30)), 1, {}
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    n = int(rng.choice([1, 7, 63, 1000, 4097, 65537, 999983, int(rng.integers(1, 3_000_000))]))
    k = int(rng.choice([0, 4, 8, 12, 32]))
    dtype = int(rng.integers(0, 2))
    return p, g, ell, n, dtype, k, ordering, schedule


@pytest.mark.parametrize("seed", range(120))
def test_random_plan_equals_oracle(seed):
    rng = np.random.default_rng(31000 + seed)
    p, g, ell, n, dtype, k, ordering, schedule = _case(rng)
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k, ordering=ordering or 2, schedule=schedule)
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, ordering=ordering, schedule=schedule)
    fl, sb, sec, p2p = B.optcc_plan_tables(plan)
    assert fl.tobytes() == oplan.flows.tobytes()
    assert np.array_equal(sb, oplan.step_begin) and np.array_equal(sec, oplan.sec_bounds) and np.array_equal(p2p, oplan.p2p_bounds)
    i = plan.info
    assert (i["k"], i["n_steps"], i["m"], i["H"], i["U_p2p"], i["construction"]) == \
           (oplan.k, oplan.n_steps, oplan.m, oplan.H, oplan.U_p2p, oplan.construction)
    if len(oplan.flows) <= 20000:
        tot = OI.check_plan(oplan)                      # exactly once, hazards, regions tile [0, n)
        assert tot["reduce_elems"] == tot["copy_elems"] == (p - 1) * n
        c = B.optcc_cost(plan)
        sim = cost_sim.simulate(oplan)
        assert abs(c["T"] - float(sim["T"])) <= 1e-12 * c["T"]
        assert c["lb_table1"] <= c["T"] * (1 + 1e-12)
