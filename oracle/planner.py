"""Canonical OPTCC plan tables, written from docs/PLAN_SPEC.md and PAPER.md §4, App. C/D/E.

Test infrastructure only (see oracle/__init__.py).  Pure Python loops; every flow is emitted by
the rule of the paper passage cited next to it, then the list is sorted as PLAN_SPEC §3 says.
"""
import math
from dataclasses import dataclass, field

import numpy as np

# PLAN_SPEC §3 enumerations
REDUCE, COPY = 0, 1
S1, S2, S3, S4, BUB_UP, BUB_DOWN, N_COLLECT, N_DISTRIBUTE = range(8)
NIC, NVLINK = 0, 1
F32, BF16 = 0, 1
C0, C1, C2, C3 = 0, 1, 2, 3
OPTCC, RING_DEGRADED = 0, 1   # PLAN_SPEC §1 option `schedule`

FLOW_DTYPE = np.dtype([
    ("off", "<u8"), ("len", "<u8"), ("step", "<u4"), ("seg", "<u4"), ("sec", "<u4"),
    ("src", "<u2"), ("dst", "<u2"), ("op", "u1"), ("stage", "u1"), ("link", "u1"), ("part", "u1"),
    ("reserved", "<u4"),
], align=False)
assert FLOW_DTYPE.itemsize == 40


class PlanError(ValueError):
    def __init__(self, code, msg):
        super().__init__(msg)
        self.code = code  # "EINVAL" | "EUNSUPPORTED"


@dataclass
class Plan:
    p: int
    g: int
    q: int
    m: int
    H: int
    k: int
    n: int
    dtype: int
    construction: int
    A: int            # elements per 16-byte unit
    U: int            # units
    U_ring: int
    U_p2p: int
    n_ring: int       # elements on the ring path
    n_p2p: int        # elements on the P2P (bubble) path
    n_steps: int
    ell: list
    stragglers: list  # straggler server indices, PLAN_SPEC §1 order
    healthy: list     # healthy server indices, server order
    flows: np.ndarray = field(repr=False, default=None)       # FLOW_DTYPE, sorted
    step_begin: np.ndarray = field(repr=False, default=None)  # u32 [n_steps+1]
    sec_bounds: np.ndarray = field(repr=False, default=None)  # u64, elements
    p2p_bounds: np.ndarray = field(repr=False, default=None)  # u64, elements
    schedule: int = 0
    ordering: int = 2


def _split(lo, hi, parts, i):
    """PLAN_SPEC §2: split(lo, hi, parts, i) on unit indices, exact integers."""
    return lo + (i * (hi - lo)) // parts


def classify(p, g, ell):
    """PLAN_SPEC §1: validate, find stragglers and the healthy ring."""
    if p < 3 or g < 1 or p % g != 0:
        raise PlanError("EINVAL", "p >= 3, g >= 1, g | p required")
    if len(ell) != p:
        raise PlanError("EINVAL", "ell must have p entries")
    for x in ell:
        if not math.isfinite(x) or x < 1.0:
            raise PlanError("EINVAL", "ell must be finite and >= 1")
    q = p // g
    for v in range(q):
        if any(ell[v * g + i] != ell[v * g] for i in range(g)):
            raise PlanError("EINVAL", "ranks of one server must share ell (PXN, :274)")
    stragglers = [v for v in range(q) if ell[v * g] > 1.0]
    stragglers.sort(key=lambda v: (-ell[v * g], v))
    healthy = [v for v in range(q) if not ell[v * g] > 1.0]
    if len(healthy) < 2:
        raise PlanError("EINVAL", "at least two healthy servers required")
    if g > 1 and len(stragglers) == 0:
        raise PlanError("EUNSUPPORTED", "g > 1 without a straggler is NCCL's multi-channel ring (:88), a comparison system")
    return q, stragglers, healthy


def p2p_units(p, ell1, U):
    """PLAN_SPEC §2 / PAPER.md:739-748: units on the P2P path, one IEEE-double rounding."""
    num = 2.0 - ell1
    den = float(p - 2) * ell1 + 2.0
    f = num / den
    x = float(U) * f
    return int(math.floor(x + 0.5))


def auto_k(construction, ell1, H, ring_units):
    """PLAN_SPEC §2 'k (R2)'."""
    if construction == C0:
        return 1
    if construction == C1:
        c = ell1 - 1.0 if ell1 < 2.0 else 1.0
    elif construction == C2:
        c = 1.0
    else:
        c = 2.0
    k_t = 4 * int(math.ceil(5.0 * c - 1e-9))
    R = ring_units * 16
    k_c = 4 * ((R // (H * 65536)) // 4)
    return max(4, min(k_t, k_c))


def build_plan(p, g, ell, n, dtype, k=0, _u_p2p_override=None, schedule=OPTCC, ordering=2):
    """optcc_plan of the oracle.  `_u_p2p_override` (brute-force search only) replaces U_p2p."""
    ell = [float(x) for x in ell]
    if schedule not in (OPTCC, RING_DEGRADED):
        raise PlanError("EINVAL", "schedule")
    if schedule == RING_DEGRADED and g != 1:
        if p >= 3 and g >= 1 and p % g == 0:
            raise PlanError("EUNSUPPORTED", "the ring baseline is defined for g = 1")
    q, stragglers, healthy = classify(p, g, ell)
    if ordering not in (1, 2, 3):
        raise PlanError("EINVAL", "ordering is 1 or 2 (:138) or 3 (the four-pattern mix, :144-155)")
    if ordering in (1, 3) and not (g == 1 and len(stragglers) == 1 and schedule == OPTCC):
        raise PlanError("EUNSUPPORTED", "ordering (1) and the mix are constructed for one straggler, g = 1 (PLAN_SPEC C1', C1'')")
    if n <= 0 or n > 2 ** 40:
        raise PlanError("EINVAL", "0 < n <= 2^40 required")
    if dtype not in (F32, BF16):
        raise PlanError("EINVAL", "dtype")
    if k != 0 and (k % 4 != 0 or k < 0 or k > 65536):
        raise PlanError("EINVAL", "k must be a multiple of 4 (:155), <= 65536")
    m, H = len(stragglers), len(healthy)
    construction = C0 if (m == 0 or schedule == RING_DEGRADED) else (C3 if g > 1 else (C1 if m == 1 else C2))
    A = 4 if dtype == F32 else 8
    U = -(-n // A)
    E = lambda u: min(u * A, n)
    ell1 = ell[stragglers[0] * g] if m else 1.0

    U_p2p = 0
    if construction == C1 and ell1 < 2.0:
        U_p2p = p2p_units(p, ell1, U)
    if construction == C1 and _u_p2p_override is not None:
        U_p2p = _u_p2p_override
    U_ring = U - U_p2p

    part_lo = [_split(0, U, g, lam) for lam in range(g + 1)]
    ring = [(0, U_ring)] if construction in (C0, C1) else [(part_lo[l], part_lo[l + 1]) for l in range(g)]
    if k == 0 or construction == C0:
        k = auto_k(construction, ell1, H, ring[0][1] - ring[0][0])
    nsec = p if construction == C0 else H

    def sec_units(lam, b, c):
        lo, hi = ring[lam]
        s0, s1 = _split(lo, hi, k, b), _split(lo, hi, k, b + 1)
        return _split(s0, s1, nsec, c), _split(s0, s1, nsec, c + 1)

    def p2p_piece(b):
        return _split(U_ring, U, k, b), _split(U_ring, U, k, b + 1)

    flows = []

    def emit(step, op, stage, link, part, src, dst, seg, sec, rng):
        off, ln = E(rng[0]), E(rng[1]) - E(rng[0])
        if ln > 0:
            flows.append((off, ln, step, seg, sec, src, dst, op, stage, link, part, 0))

    if construction == C1 and ordering == 3:
        # C1'': the four-pattern mix of :144-155 (PLAN_SPEC §4 C1'').  A, C: ordering (1); B, D: ordering (2); one
        # stage per parallel body (2(p-1) slots per stage, :146); A and B start in body 4γ, C and D one body later, so a
        # group of four segments spans five bodies and the schedule has k+1 bodies (:155, :169).
        n_steps = (k + 1) * H
        sg = stragglers[0]
        hr = list(healthy)
        bubbles = ell1 < 2.0
        W = lambda j, t: t if t < j else t + 1          # ring link j idle in window j
        for b in range(k):
            gam, pat = divmod(b, 4)
            s0 = 4 * gam + (1 if pat >= 2 else 0)       # first body of the segment
            if pat in (0, 2):                           # patterns A, C: S1 -> S2 -> S3 -> S4 (:148, :150)
                for j in range(H):
                    for t in range(H - 1):
                        c = (j - t) % H
                        emit(s0 * H + W(j, t), REDUCE, S1, NIC, 0, hr[j], hr[(j + 1) % H], b, c, sec_units(0, b, c))
                        emit((s0 + 3) * H + W(j, t), COPY, S4, NIC, 0, hr[j], hr[(j + 1) % H], b, c, sec_units(0, b, c))
                for a in range(H):
                    d = (a + 1) % H
                    # the straggler adds its own data to the uploaded partial sum (:130-132) ...
                    emit((s0 + 1) * H + a, REDUCE, S2, NIC, 0, hr[a], sg, b, (a + 1) % H, sec_units(0, b, (a + 1) % H))
                    # ... and returns the global sum to the uploader's ring successor (:132, R11)
                    emit((s0 + 2) * H + a, COPY, S3, NIC, 0, sg, hr[d], b, d, sec_units(0, b, d))
            else:                                       # patterns B, D: S3 -> S1 -> S4 -> S2 (:149, :151)
                for a in range(H):
                    d = (a + 1) % H
                    # the straggler's raw section is folded in at its owner first (:138 ordering (2)) ...
                    emit(s0 * H + a, REDUCE, S3, NIC, 0, sg, hr[d], b, (d + 1) % H, sec_units(0, b, (d + 1) % H))
                    # ... and the owner sends the global sum back last
                    emit((s0 + 3) * H + a, COPY, S2, NIC, 0, hr[a], sg, b, (a + 1) % H, sec_units(0, b, (a + 1) % H))
                for j in range(H):
                    for t in range(H - 1):
                        emit((s0 + 1) * H + W(j, t), REDUCE, S1, NIC, 0, hr[j], hr[(j + 1) % H], b, (j - t) % H,
                             sec_units(0, b, (j - t) % H))
                        emit((s0 + 2) * H + W(j, t), COPY, S4, NIC, 0, hr[j], hr[(j + 1) % H], b, (j + 1 - t) % H,
                             sec_units(0, b, (j + 1 - t) % H))
            if bubbles:                                 # bubble-up in body b, bubble-down in body b+1, as in C1 (:165)
                for a in range(H):
                    emit(b * H + a, REDUCE, BUB_UP, NIC, 0, hr[a], sg, b, 0, p2p_piece(b))
                    emit((b + 1) * H + a, COPY, BUB_DOWN, NIC, 0, sg, hr[(a + 1) % H], b, 0, p2p_piece(b))
    elif construction == C1 and ordering == 1:
        # C1': ordering (1) of :138, S1 -> S2 -> S3 -> S4, one stage per body (PLAN_SPEC §4 C1')
        n_steps = (k + 3) * H
        sg = stragglers[0]
        hr = list(healthy)
        bubbles = ell1 < 2.0
        W = lambda j, t: t if t < j else t + 1          # ring link j idle in window j
        for B in range(k + 3):
            base = B * H
            for j in range(H):
                src, dst = hr[j], hr[(j + 1) % H]
                for t in range(H - 1):
                    step = base + W(j, t)
                    if B < k:            # Stage 1 hop t of segment B: healthy-only partial sums (:126)
                        c = (j - t) % H
                        emit(step, REDUCE, S1, NIC, 0, src, dst, B, c, sec_units(0, B, c))
                    if 3 <= B:           # Stage 4 hop t of segment B-3: global sum of section j starts at healthy j (:136)
                        c = (j - t) % H
                        emit(step, COPY, S4, NIC, 0, src, dst, B - 3, c, sec_units(0, B - 3, c))
            for a in range(H):
                d = (a + 1) % H
                step = base + a
                if 1 <= B <= k:          # Stage 2: owner a uploads its partial sum, the straggler adds its own (:130-132)
                    c = (a + 1) % H
                    emit(step, REDUCE, S2, NIC, 0, hr[a], sg, B - 1, c, sec_units(0, B - 1, c))
                if 2 <= B <= k + 1:      # Stage 3: the straggler returns the global sum to the uploader's successor (:132, R11)
                    emit(step, COPY, S3, NIC, 0, sg, hr[d], B - 2, d, sec_units(0, B - 2, d))
                if bubbles and B < k:    # bubble-up / bubble-down as in C1 (:165)
                    emit(step, REDUCE, BUB_UP, NIC, 0, hr[a], sg, B, 0, p2p_piece(B))
                if bubbles and 1 <= B <= k:
                    emit(step, COPY, BUB_DOWN, NIC, 0, sg, hr[d], B - 1, 0, p2p_piece(B - 1))
    elif construction == C0:
        # plain ring reduce-scatter + allgather over all p ranks (:52, :72)
        n_steps = 2 * (p - 1)
        for t in range(p - 1):
            for j in range(p):
                d = (j + 1) % p
                emit(t, REDUCE, S1, NIC, 0, j, d, 0, (j - t) % p, sec_units(0, 0, (j - t) % p))
                emit(p - 1 + t, COPY, S4, NIC, 0, j, d, 0, (j + 1 - t) % p, sec_units(0, 0, (j + 1 - t) % p))
    else:
        nstr = m                       # stragglers seen by the NIC schedule
        P = H + nstr - 1               # windows per body: H (C1/C3) or p-1 (C2, :788)
        if construction == C3:
            D = 1 + -(-(g - 2) // P)
            n_steps = (k + D + 2) * P + g - 2
        else:
            D = 0
            n_steps = (k + 1) * P
        bubbles = construction == C1 and (ell1 < 2.0 or _u_p2p_override is not None)
        for lam in range(g):
            hr = [v * g + lam for v in healthy]         # leaders of the healthy servers (:854)
            sr = [v * g + lam for v in stragglers]
            W = lambda j, t: t if t < j else t + nstr   # ring link j idle in windows [j, j+m)
            for B in range(k + 1):                      # C1/C2 body index
                base = (B + D) * P
                for j in range(H):
                    src, dst = hr[j], hr[(j + 1) % H]
                    for t in range(H - 1):
                        step = base + W(j, t)
                        if B < k:       # Stage 1 hop t of segment B (:126)
                            c = (j - t) % H
                            emit(step, REDUCE, S1, NIC, lam, src, dst, B, c, sec_units(lam, B, c))
                        if B >= 1:      # Stage 4 hop t of segment B-1 (:136)
                            c = (j + 1 - t) % H
                            emit(step, COPY, S4, NIC, lam, src, dst, B - 1, c, sec_units(lam, B - 1, c))
                for i, sg in enumerate(sr):
                    for a in range(H):
                        w = a + i
                        d = (a + 1) % H
                        step = base + w
                        if B >= 1:      # Stage 2: owner a sends the global sum to the straggler (:130, :138 ordering 2)
                            c = (a + 1) % H
                            emit(step, COPY, S2, NIC, lam, hr[a], sg, B - 1, c, sec_units(lam, B - 1, c))
                        if B < k:       # Stage 3: straggler's raw section into its owner d (:132, :138 ordering 2)
                            c = (d + 1) % H
                            emit(step, REDUCE, S3, NIC, lam, sg, hr[d], B, c, sec_units(lam, B, c))
                        if bubbles and B < k:    # bubble-up: healthy a's raw P2P piece into the straggler (:165, R9)
                            emit(step, REDUCE, BUB_UP, NIC, lam, hr[a], sg, B, 0, p2p_piece(B))
                        if bubbles and B >= 1:   # bubble-down: straggler's P2P result to d (:165)
                            emit(step, COPY, BUB_DOWN, NIC, lam, sg, hr[d], B - 1, 0, p2p_piece(B - 1))
            if construction == C3:
                for v in range(q):
                    for b in range(k):
                        for c in range(H):
                            rng = sec_units(lam, b, c)
                            for h in range(g - 1):
                                # collect on the backward local ring, leader only receives (:862, :875, :894)
                                emit(b * P + c + h, REDUCE, N_COLLECT, NVLINK, lam,
                                     v * g + (lam - 1 - h) % g, v * g + (lam - 2 - h) % g, b, c, rng)
                                # distribute on the forward local ring, leader sends first (:863, :876, :894)
                                emit((b + D + 2) * P + c + h, COPY, N_DISTRIBUTE, NVLINK, lam,
                                     v * g + (lam + h) % g, v * g + (lam + h + 1) % g, b, c, rng)

    arr = np.array(flows, dtype=FLOW_DTYPE) if flows else np.zeros(0, dtype=FLOW_DTYPE)
    order = np.lexsort((arr["off"], arr["dst"], arr["src"], arr["stage"], arr["link"], arr["step"]))
    arr = arr[order]
    step_begin = np.searchsorted(arr["step"], np.arange(n_steps + 1), side="left").astype(np.uint32)

    sb = []
    for lam in range(g if construction in (C2, C3) else 1):
        for b in range(k):
            for c in range(nsec):
                sb.append(E(sec_units(lam, b, c)[0]))
    sb.append(E(ring[-1][1]))
    pb = [E(p2p_piece(b)[0]) for b in range(k)] + [E(U)] if (construction == C1 and ell1 < 2.0) else []

    return Plan(p=p, g=g, q=q, m=m, H=H, k=k, n=n, dtype=dtype, construction=construction, A=A, U=U,
                U_ring=U_ring, U_p2p=U_p2p, n_ring=E(U_ring), n_p2p=n - E(U_ring), n_steps=n_steps,
                ell=ell, stragglers=stragglers, healthy=healthy, flows=arr, step_begin=step_begin,
                sec_bounds=np.array(sb, dtype=np.uint64), p2p_bounds=np.array(pb, dtype=np.uint64), schedule=schedule, ordering=ordering)
