"""Brute-force minimisation of completion time over chunk splits for p <= 5 (north_star).

The planner's P2P share (PLAN_SPEC §2) must be the split that an exhaustive search
over all integer splits finds; the fluid optimum must equal Theorem 6 (:413-455)."""
from fractions import Fraction as Fr

import pytest

from oracle import brute_force, closed_forms as cf
from oracle import planner as P


@pytest.mark.parametrize("p", [3, 4, 5])
@pytest.mark.parametrize("ell", [8.0 / 7.0, 1.25, 4.0 / 3.0, 1.5, 1.75])
def test_split_search_small_ell(p, ell):
    k = 4
    U = k * 240                     # 240 units per segment
    n = 4 * U
    res = brute_force.search_p2p_split(p, ell, n, k, step=1, check=False)
    planner_choice = P.build_plan(p, 1, [ell] + [1.0] * (p - 1), n, P.F32, k=k).U_p2p
    closed = cf.p2p_fraction(p, ell) * U
    assert abs(planner_choice - closed) <= Fr(1, 2)
    # fluid objective (max port load): minimum is Theorem 6, attained within one unit of the closed form
    # (sections are floor-split, so port loads wobble by up to k(p-1) units around the divisible case)
    best, arg = brute_force.argmin(res, 2)
    assert min(abs(a - closed) for a in arg) <= k * (p - 1)
    lb = cf.lb_thm6(p, ell, n)
    assert lb <= best <= lb * (1 + Fr(2 * k * (p - 1), U))
    # finite-k simulated T: the planner's split is within 1.5 % of the best split found by exhaustive search
    bestT, argT = brute_force.argmin(res, 1)
    chosenT = next(r[1] for r in res if r[0] == planner_choice)
    assert bestT <= chosenT <= bestT * Fr(1015, 1000)
    assert chosenT >= cf.lb_thm6(p, ell, n)


@pytest.mark.parametrize("p", [4, 5])
@pytest.mark.parametrize("ell", [2.0, 3.0])
def test_split_search_large_ell_prefers_no_p2p(p, ell):
    # :171 l >= 2 straggler-bottlenecked: any data on the P2P path only loads the straggler link more. Config C1.
    k = 4
    n = 4 * k * 60
    res = brute_force.search_p2p_split(p, ell, n, k, step=1, check=False)
    best, arg = brute_force.argmin(res, 2)
    assert arg == [0] and best == cf.lb_thm6(p, ell, n) == Fr(ell) * n
    bestT, argT = brute_force.argmin(res, 1)
    assert 0 in argT and bestT == cf.T_eq1(p, ell, k, n)
    assert P.build_plan(p, 1, [ell] + [1.0] * (p - 1), n, P.F32, k=k).U_p2p == 0


def test_every_searched_split_is_still_a_correct_allreduce():
    res = brute_force.search_p2p_split(4, 1.5, 4 * 4 * 30, 4, step=7, check=True)
    assert len(res) > 10


@pytest.mark.parametrize("p,ell,den", [(5, 1.5, 13), (3, 1.5, 7), (4, 1.5, 10), (5, 1.25, 23)])
def test_split_search_divisible_case_is_exactly_the_closed_form(p, ell, den):
    # when s' (:748) and (2-l)s'/l (:744) are whole units the exhaustive argmin IS the closed form,
    # the fluid minimum IS Theorem 6 and the simulated minimum IS Eq.(2)
    k = 4
    U = den * k * (p - 1)
    n = 4 * U
    res = brute_force.search_p2p_split(p, ell, n, k, step=1, check=False)
    closed = cf.p2p_fraction(p, ell) * U
    assert closed.denominator == 1
    best, arg = brute_force.argmin(res, 2)
    assert arg == [int(closed)] and best == cf.lb_thm6(p, ell, n)
    bestT, argT = brute_force.argmin(res, 1)
    assert int(closed) in argT and bestT == cf.T_eq2(p, ell, k, n)
