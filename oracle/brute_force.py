"""Brute-force search over chunk splits for p <= 5 (BASELINE.json north_star; SURVEY §8(c) pins).

Test infrastructure only (see oracle/__init__.py).  For a small n every admissible P2P share
U_p2p in {0, .., U} is tried: the plan is rebuilt with that split, checked (exactly-once), and its
completion time simulated.  Two objectives are returned per split:
  T      event-simulated completion time of the finite-k plan
  fluid  max over NIC ports of the time-weighted load (the k -> infinity body bound; the quantity the
         proof of Theorem 6 minimises, :432-455)
"""
from . import planner as P
from . import cost_sim
from . import interpreter


def search_p2p_split(p, ell_straggler, n, k, straggler=0, dtype=P.F32, step=1, check=True):
    """Returns list of (U_p2p, T, fluid) for U_p2p = 0, step, 2 step, ... <= U (all k pieces non-empty or zero)."""
    assert p <= 5, "brute force is for tiny p only"
    ell = [1.0] * p
    ell[straggler] = float(ell_straggler)
    A = 4 if dtype == P.F32 else 8
    U = -(-n // A)
    out = []
    for up in range(0, U + 1, step):
        if U - up < 1:
            continue
        plan = P.build_plan(p, 1, ell, n, dtype, k=k, _u_p2p_override=up)
        if check:
            interpreter.check_plan(plan)
        sim = cost_sim.simulate(plan)
        out.append((up, sim["T"], sim["fluid"]))
    return out


def argmin(results, key):
    """All U_p2p attaining the minimum of column `key` (1 = T, 2 = fluid)."""
    best = min(r[key] for r in results)
    return best, [r[0] for r in results if r[key] == best]
