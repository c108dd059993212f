"""Closed forms printed in PAPER.md, in exact rationals (fractions.Fraction).

Test infrastructure only (see oracle/__init__.py).  Every function cites the passage it restates.
All times are in "element-times" (a healthy NIC moves one element per unit).
"""
from fractions import Fraction as Fr


def _fr(x):
    """Exact rational value of an int / float / Fraction (a double is a binary rational)."""
    return x if isinstance(x, Fr) else Fr(x)


def T0(p, n, g=1):
    """Fault-free optimum T0 = 2(p-1)n/(g p)  (the printed 'q' is the g of :68, R6)."""
    return Fr(2 * (p - 1) * n, g * p)


def T0_server(p, n, g):
    """Server-ring base 2(q-1)n/(q g) that the series of Theorem 3 (:112) are relative to (R6)."""
    q = p // g
    return Fr(2 * (q - 1) * n, q * g)


def lb_thm1(p, ell, n=1):
    """Theorem 1 (:76, :338): T >= max{2l(p-1)/(l(p-1)+1), l} n."""
    l = _fr(ell)
    return max(2 * l * (p - 1) / (l * (p - 1) + 1), l) * n


def thm1_switch(p):
    """Regime switch of Theorem 1 / Table 1: l = 2 - 1/(p-1)  (:19, :393-403)."""
    return 2 - Fr(1, p - 1)


def lb_thm2(p, ells, n=1):
    """Theorem 2 (:82, :473): T >= max{2(p-1)/(p-m+sum 1/l_i), l_1} n, l_1 = max l_i."""
    ls = [_fr(l) for l in ells]
    m = len(ls)
    y0 = Fr(2 * (p - 1)) / (p - m + sum(1 / l for l in ls))
    return max(y0, max(ls)) * n


def y0_thm2(p, ells):
    """y0 of Theorem 2's proof (:503) and x_i* = y0 / l_i (:505)."""
    ls = [_fr(l) for l in ells]
    return Fr(2 * (p - 1)) / (p - len(ls) + sum(1 / l for l in ls))


def lb_thm3(p, g, ell, n=1):
    """Theorem 3 (:538): T >= (n/g) max{2l(q-1)/(1+l(q-1)), l}; the :112 display equals it with p-g=g(q-1)."""
    l = _fr(ell)
    q = p // g
    return Fr(n, g) * max(2 * l * (q - 1) / (1 + l * (q - 1)), l)


def lb_thm3_display(p, g, ell, n=1):
    """Theorem 3 as displayed at :112: max{2l(p-g)/(g(l(p-g)+g)), l/g} n."""
    l = _fr(ell)
    return max(2 * l * (p - g) / (g * (l * (p - g) + g)), l / g) * n


def lb_thm6(p, ell, n=1):
    """Theorem 6, tight single-straggler bound (:413): T >= max{2l(p-1)/(l(p-2)+2), l} n."""
    l = _fr(ell)
    return max(2 * l * (p - 1) / (l * (p - 2) + 2), l) * n


def zstar_thm6(p, ell):
    """z* = 2(p-1)/(l(p-2)+2): straggler sends and receives z* n elements at the optimum (:455)."""
    l = _fr(ell)
    return Fr(2 * (p - 1)) / (l * (p - 2) + 2)


def lb_thm13(p, g, ell, n=1):
    """Theorem 13, tight multi-GPU bound (:664): T >= (n/g) max{2l(q-1)/(l(q-2)+2), l}."""
    l = _fr(ell)
    q = p // g
    return Fr(n, g) * max(2 * l * (q - 1) / (l * (q - 2) + 2), l)


def series_thm1_small(p, ell):
    """Table 1 small-l series, first-order part: 1 + (l-1)/(l p)  [x T0]  (:22)."""
    l = _fr(ell)
    return 1 + (l - 1) / (l * p)


def series_large(p, ell):
    """Table 1 large-l series, first-order part: l/2 + l/(2p)  [x T0]  (:22-24)."""
    l = _fr(ell)
    return l / 2 + l / (2 * p)


def series_thm2_small(p, ells):
    """Table 1 row 3 small-l series: 1 + sum((l_i-1)/l_i)/p  [x T0]  (:23)."""
    return 1 + sum((_fr(l) - 1) / _fr(l) for l in ells) / p


def series_thm3_small(p, g, ell):
    """Table 1 row 4 small-l series: 1 + g(l-1)/(l p)  [x T0_server, see R6]  (:24, :112)."""
    l = _fr(ell)
    return 1 + g * (l - 1) / (l * p)


def section_size(p, k, n):
    """s = n/(k(p-1))  (:124, :169)."""
    return Fr(n, k * (p - 1))


def section_size_bubble(p, k, ell, n):
    """s' = n l / (k[(p-2)l + 2])  (:748)."""
    l = _fr(ell)
    return n * l / (k * ((p - 2) * l + 2))


def p2p_per_segment(p, k, ell, n):
    """P2P path per segment: (2-l) s'/l elements (:739-746, R8)."""
    l = _fr(ell)
    return (2 - l) * section_size_bubble(p, k, l, n) / l


def p2p_fraction(p, ell):
    """Share of n on the P2P path: k (2-l)s'/l / n = (2-l)/((p-2)l+2)  (from :746-748)."""
    l = _fr(ell)
    return (2 - l) / ((p - 2) * l + 2)


def T_eq1(p, ell, k, n):
    """Eq.(1) (:173): T = l n (k+1)/k, l >= 2."""
    return _fr(ell) * n * Fr(k + 1, k)


def T_eq2(p, ell, k, n):
    """Eq.(2) (:185, :752): T = 2(p-1) l n/((p-2)l+2) (k+l-1)/k, l < 2."""
    l = _fr(ell)
    return 2 * (p - 1) * l * n / ((p - 2) * l + 2) * (k + l - 1) / k


def T_single(p, ell, k, n):
    """Single-straggler time: Eq.(2) for l < 2, Eq.(1) for l >= 2 (:171-185)."""
    return T_eq2(p, ell, k, n) if _fr(ell) < 2 else T_eq1(p, ell, k, n)


def T_single_limit(p, ell, n=1):
    """k -> infinity limits of Eq.(1)/(2) (:173, :185)."""
    l = _fr(ell)
    return 2 * (p - 1) * l * n / ((p - 2) * l + 2) if l < 2 else l * n


def overhead_single_small(p, ell):
    """T/T0 = p l/((p-2)l+2) for l in [1,2], at most 1 + 1/(p-1)  (:760-762)."""
    l = _fr(ell)
    return p * l / ((p - 2) * l + 2)


def T_body_multi(p, ells, k, n):
    """D.3 (:805): T_body = max{2(p-1)s, (l_1(p-m)+2(m-1))s}, s = n/(k(p-m))."""
    ls = [_fr(l) for l in ells]
    m = len(ls)
    s = Fr(n, k * (p - m))
    return max(2 * (p - 1) * s, (max(ls) * (p - m) + 2 * (m - 1)) * s)


def T_multi_paper(p, ells, k, n):
    """D.3 (:809): T = (k+4) T_body (the paper's own pipeline; an upper bound for the canonical plan)."""
    return (k + 4) * T_body_multi(p, ells, k, n)


def T_multi_limit(p, ells, n=1):
    """(:831): max{2(p-1)/(p-m), l_1 + 2(m-1)/(p-m)} n."""
    ls = [_fr(l) for l in ells]
    m = len(ls)
    return max(Fr(2 * (p - 1), p - m), max(ls) + Fr(2 * (m - 1), p - m)) * n


def T_multigpu_bound(p, g, ell, k, n):
    """Eq.(21)/(22) (:920, :926): T <= max{l,2} n (k+5.5)/(g k)."""
    l = _fr(ell)
    return max(l, Fr(2)) * n * (2 * k + 11) / (2 * g * k)


def T_multigpu_limit(p, g, ell, n=1):
    """k -> infinity of Eq.(21)/(22): max{l,2} n/g."""
    return max(_fr(ell), Fr(2)) * Fr(n, g)


def T_r2ccl(p, ell, n=1):
    """R2CCL closed form used by the paper for plotting (:963): T_NCCL (1 + p(l-1)/(2(p-1)))."""
    l = _fr(ell)
    return T0(p, n) * (1 + p * (l - 1) / (2 * (p - 1)))


def T_ring_degraded(p, ells, n=1):
    """Plain ring on the degraded topology (the ICCL comparison point, :199, :217) under the bandwidth model: every
    one of the 2(p-1) ring steps moves n/p elements over every link and waits for the slowest one: max(l) T0."""
    return max([_fr(l) for l in ells] + [Fr(1)]) * T0(p, n)


def T_multigpu_multi_composed(p, g, ells, k, n):
    """m >= 2 straggler servers with g GPUs each: NOT from the paper (E.5 :943 omits it).  Composition of D.3's body
    max{2(q-1), l_1(q-m) + 2(m-1)} s (:805) on the n/g elements of one leader cycle with E.4's body count k + 5.5
    (:916); an upper-bound form for the canonical composed plan, checked against the event simulation only."""
    ls = [_fr(l) for l in ells]
    m, q = len(ls), p // g
    body = max(Fr(2 * (q - 1)), max(ls) * (q - m) + 2 * (m - 1)) / (q - m)
    return Fr(n, g) * body * Fr(2 * k + 11, 2 * k)
