"""Pins for oracle/closed_forms.py against what the paper prints and what the mathematics fixes.

A pin never re-types the formula under test: it checks it against a *different* statement of the same
fact (a proof step, a series, a limit, a special case, a printed number, a brute-force minimisation).
"""
from fractions import Fraction as Fr

import pytest

from oracle import closed_forms as cf

PS = [3, 4, 5, 8, 16, 32, 64, 128, 1024]
ELLS = [Fr(8, 7), Fr(4, 3), Fr(3, 2), Fr(8, 5), Fr(2), Fr(3)]


def test_T0_is_ring_allreduce_volume_over_p_links():
    # :52 "each GPU sending and receiving approximately twice the message size": ring RS+AG moves
    # (p-1) chunks of n/p per GPU twice over a unit-rate link.
    for p in PS:
        n = 7 * p
        assert cf.T0(p, n) == 2 * (p - 1) * Fr(n, p)
        # g>1: g concurrent channels each carrying n/g (fn.3 :88)
        for g in (2, 4, 8):
            if p % g == 0:
                assert cf.T0(p, n, g) == cf.T0(p, n) / g


def _minmax_1d(branch_dec, branch_inc, lo=Fr(1), hi=Fr(4), steps=3000):
    """Brute-force min over z >= 1 of max(two branches) on a fine rational grid (proof steps :383, :451)."""
    best = None
    for i in range(steps + 1):
        z = lo + (hi - lo) * Fr(i, steps)
        v = max(branch_dec(z), branch_inc(z))
        best = v if best is None or v < best else best
    return best


@pytest.mark.parametrize("p", [3, 5, 16])
@pytest.mark.parametrize("ell", ELLS)
def test_thm1_is_the_minmax_of_its_proof(p, ell):
    # :383  T/n >= min_{z>=1} max{2 - z/(p-1), l z}
    grid = _minmax_1d(lambda z: 2 - z / (p - 1), lambda z: ell * z)
    exact = cf.lb_thm1(p, ell)
    assert exact <= grid <= exact * Fr(1001, 1000)


@pytest.mark.parametrize("p", [3, 5, 16])
@pytest.mark.parametrize("ell", ELLS)
def test_thm6_is_the_minmax_of_its_proof(p, ell):
    # :451  T/n >= min_{z>=1} max{2 + (l-2)z/(p-1), l z}
    grid = _minmax_1d(lambda z: 2 + (ell - 2) * z / (p - 1), lambda z: ell * z)
    exact = cf.lb_thm6(p, ell)
    assert exact <= grid <= exact * Fr(1001, 1000)


def test_thm6_zstar_solves_the_intersection():
    # :453-455: 2 + (l-2) z/(p-1) = l z at z*
    for p in PS:
        for ell in ELLS:
            if ell <= 2:
                z = cf.zstar_thm6(p, ell)
                assert 2 + (ell - 2) * z / (p - 1) == ell * z
                assert z >= 1
                assert cf.lb_thm6(p, ell) == ell * z


def test_regime_switches():
    for p in PS:
        sw = cf.thm1_switch(p)
        # both branches of Theorem 1 meet exactly at l = 2 - 1/(p-1)  (:393-403)
        assert 2 * sw * (p - 1) / (sw * (p - 1) + 1) == sw
        assert cf.lb_thm1(p, sw) == sw
        # below the switch the first branch wins, above it the second
        assert cf.lb_thm1(p, sw - Fr(1, 100)) > sw - Fr(1, 100)
        assert cf.lb_thm1(p, sw + Fr(1, 100)) == sw + Fr(1, 100)
        # Theorem 6 / 13 switch at l = 2 (:453, :705; Table 2 note 1 :292)
        assert 2 * Fr(2) * (p - 1) / (2 * (p - 2) + 2) == 2
        assert cf.lb_thm6(p, Fr(2)) == 2
        assert cf.lb_thm6(p, Fr(21, 10)) == Fr(21, 10)


def test_thm6_sharpens_thm1_and_thm13_sharpens_thm3():
    for p in PS:
        for ell in ELLS:
            assert cf.lb_thm6(p, ell) >= cf.lb_thm1(p, ell)       # :409 "strictly stronger"
            for g in (2, 4, 8):
                if p % g == 0 and p // g >= 3:
                    assert cf.lb_thm13(p, g, ell) >= cf.lb_thm3(p, g, ell)   # :660


def test_consistency_reductions():
    for p in PS:
        for ell in ELLS:
            assert cf.lb_thm2(p, [ell]) == cf.lb_thm1(p, ell)          # :84, :526  m=1
            assert cf.lb_thm3(p, 1, ell) == cf.lb_thm1(p, ell)         # :114      g=1
            assert cf.lb_thm13(p, 1, ell) == cf.lb_thm6(p, ell)        # g=1
            for g in (2, 4):
                if p % g == 0:
                    assert cf.lb_thm3(p, g, ell, 5) == cf.lb_thm3_display(p, g, ell, 5)   # :112 vs :538


def test_thm2_balanced_point():
    # :505  with x_i = y0/l_i all m+1 terms of g are equal to y0
    p, ells = 64, [Fr(2), Fr(4, 3), Fr(8, 7)]
    y0 = cf.y0_thm2(p, ells)
    xs = [y0 / l for l in ells]
    assert all(l * x == y0 for l, x in zip(ells, xs))
    assert (2 * (p - 1) - sum(xs)) / (p - len(ells)) == y0
    # config C3: y0 = 1.99604 < l_1 = 2 so the l_1 branch binds
    assert y0 < 2 and cf.lb_thm2(p, ells) == 2
    assert abs(float(y0) - 1.99604) < 1e-5


@pytest.mark.parametrize("p", [64, 128, 1024])
def test_table1_series_agree_to_second_order(p):
    # Table 1 (:19-24): the printed series equal the exact bounds up to O(1/p^2) [O(g^2/p^2)]
    for ell in [Fr(8, 7), Fr(4, 3), Fr(3, 2)]:
        exact = cf.lb_thm1(p, ell, 1) / cf.T0(p, 1)
        assert abs(exact - cf.series_thm1_small(p, ell)) < Fr(4, p * p)
        ells = [ell, Fr(8, 7)]
        exact2 = cf.lb_thm2(p, ells, 1) / cf.T0(p, 1)
        assert abs(exact2 - cf.series_thm2_small(p, ells)) < Fr(8, p * p)
        for g in (4, 8):
            # R6: the Theorem-3 series (:112) is relative to 2(q-1)n/(qg)
            exact3 = cf.lb_thm3(p, g, ell, 1) / cf.T0_server(p, 1, g)
            assert abs(exact3 - cf.series_thm3_small(p, g, ell)) < Fr(4 * g * g, p * p)
    for ell in [Fr(2), Fr(3)]:
        exact = cf.lb_thm1(p, ell, 1) / cf.T0(p, 1)
        assert abs(exact - cf.series_large(p, ell)) < Fr(4, p * p)


def test_bubble_section_size_from_its_data_accounting():
    # :746  n = k[(p-1)s' + (2-l)s'/l]  and the enlarged flow lasts (1+(2-l)/l) l s' = 2 s' (:739)
    for p in PS:
        for ell in [Fr(8, 7), Fr(4, 3), Fr(3, 2), Fr(8, 5)]:
            for k in (4, 8):
                n = 1000
                s = cf.section_size_bubble(p, k, ell, n)
                assert k * ((p - 1) * s + (2 - ell) * s / ell) == n
                assert cf.p2p_per_segment(p, k, ell, n) == (2 - ell) * s / ell
                assert ell * (s + cf.p2p_per_segment(p, k, ell, n)) == 2 * s
                assert cf.p2p_fraction(p, ell) * n == k * cf.p2p_per_segment(p, k, ell, n)
                # Eq.(2) = [2k + 2(l-1)](p-1)s'  (:752)
                assert cf.T_eq2(p, ell, k, n) == (2 * k + 2 * (ell - 1)) * (p - 1) * s


def test_eq1_from_body_count():
    # :171  k+1 bodies of l(p-1)s with s = n/(k(p-1))
    for p in PS:
        for ell in [Fr(2), Fr(3)]:
            for k in (4, 8, 20):
                assert cf.T_eq1(p, ell, k, 840) == (k + 1) * ell * (p - 1) * cf.section_size(p, k, 840)


def test_special_cases_printed_in_the_paper(golden):
    for p in PS:
        assert cf.T_single_limit(p, Fr(1), 1) / cf.T0(p, 1) == golden["eq2_at_l1_over_T0"]     # :187
        assert cf.T_single_limit(p, Fr(2), 1) == golden["eq2_at_l2_over_n"]                     # :187
        for ell in [Fr(1), Fr(8, 7), Fr(3, 2), Fr(2)]:
            r = cf.overhead_single_small(p, ell)
            assert r == cf.T_single_limit(p, ell, 1) / cf.T0(p, 1)                              # :760
            assert r <= 1 + Fr(1, p - 1)                                                        # :762
        assert cf.overhead_single_small(p, Fr(2)) == 1 + Fr(1, p - 1)
        # Eq.(2)'s limit meets Theorem 6 (":756 achieves bandwidth optimality without p -> inf")
        for ell in [Fr(8, 7), Fr(3, 2)]:
            assert cf.T_single_limit(p, ell, 1) == cf.lb_thm6(p, ell, 1)
        assert cf.T_single_limit(p, Fr(3), 1) == cf.lb_thm1(p, Fr(3), 1)                        # :173
    # "less than 1% at p=128" (:36)
    p = int(golden["overhead_below_1pct_at_p"])
    assert cf.lb_thm1(p, cf.thm1_switch(p)) / cf.T0(p, 1) - 1 < Fr(1, 100)
    # 2 of 8 NICs lost -> l = 8/6 (:44); 1 of 8 -> 12.5 % (:11)
    assert abs(float(Fr(8, 6)) - golden["nic_loss_2_of_8_ell"]) < 1e-15
    assert 1 - Fr(7, 8) == Fr(golden["nic_loss_1_of_8_bw_cut"])
    # R2CCL "up to 57%" at 50% loss: closed form :963 at the smallest 8-GPU ring
    assert round(float(cf.T_r2ccl(8, 2) / cf.T0(8, 1) - 1), 2) == golden["r2ccl_overhead_50pct_loss_max"]


def test_multistraggler_and_multigpu_forms(golden):
    p, ells, n = 64, [Fr(2), Fr(4, 3), Fr(8, 7)], 61 * 8 * 100
    for k in (4, 8):
        tb = cf.T_body_multi(p, ells, k, n)
        assert cf.T_multi_paper(p, ells, k, n) == (k + golden["multistraggler_body_extra"]) * tb
    # :831 limit, config C3: 64/61 T0-relative = 1.04918
    lim = cf.T_multi_limit(p, ells, 1)
    assert lim == max(Fr(2 * 63, 61), 2 + Fr(4, 61))
    assert abs(float(lim / cf.T0(p, 1)) - 1.04918) < 1e-5
    # Eq.(21)/(22) (:920-926) and T/T_LB = (l(q-2)+2)/(l(q-1)) < q/(q-1) (:935)
    for q in (4, 16):
        for g in (4, 8):
            pp = q * g
            for ell in [Fr(8, 7), Fr(3, 2)]:
                ratio = cf.T_multigpu_limit(pp, g, ell, 1) / cf.lb_thm13(pp, g, ell, 1)
                assert ratio == (ell * (q - 2) + 2) / (ell * (q - 1))
                assert ratio < Fr(q, q - 1)
            assert cf.T_multigpu_limit(pp, g, Fr(3), 1) == cf.lb_thm13(pp, g, Fr(3), 1)   # :922 optimal
            k = 24
            assert cf.T_multigpu_bound(pp, g, Fr(2), k, 7) == 2 * Fr(7, g) * (k + Fr(golden["multigpu_body_bound_extra"])) / k


def test_baseline_md_config_values():
    # BASELINE.md §2 (k -> infinity, relative to T0 = 2(p-1)n/(gp))
    t = lambda p, g=1: cf.T0(p, 1, g)
    assert cf.lb_thm1(4, 2) / t(4) == Fr(4, 3) == cf.T_single_limit(4, 2) / t(4)
    assert abs(float(cf.lb_thm1(16, Fr(8, 7)) / t(16)) - 1.00787) < 1e-5
    assert abs(float(cf.lb_thm6(16, Fr(8, 7)) / t(16)) - 1.01587) < 1e-5
    assert abs(float(cf.lb_thm3(128, 8, 2) / t(128, 8)) - 1.00787) < 1e-5
    assert abs(float(cf.lb_thm3(128, 8, 2) / cf.T0_server(128, 1, 8)) - 1.06667) < 1e-5
    want_lb = [1, 1.00392, 1.00787, 1.01186, 1.01561, 1.03226, 1.54839]
    want_t = [1, 1.00787, 1.01587, 1.02400, 1.03171, 1.03226, 1.54839]
    ells = [Fr(1), Fr(8, 7), Fr(4, 3), Fr(8, 5), 2 - Fr(1, 31), Fr(2), Fr(3)]
    for ell, a, b in zip(ells, want_lb, want_t):
        assert abs(float(cf.lb_thm1(32, ell) / t(32)) - a) < 1e-5
        assert abs(float(cf.T_single_limit(32, ell) / t(32)) - b) < 1e-5
