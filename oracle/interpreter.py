"""Plan interpreter of the oracle: walks the flow table step by step (§4.1, :68).

Test infrastructure only (see oracle/__init__.py).  Three independent walks over the same table:
  check_plan       contributor sets per (rank, region), hazards per step, traffic sums (PLAN_SPEC §5)
  element_masks    per-element contributor bitmask arrays (what the GPU verifier must reproduce)
  run_f32/run_bf16 the arithmetic itself, one IEEE add per element per reduce flow, in table order
"""
import numpy as np

from . import planner as P


class PlanViolation(AssertionError):
    pass


def check_plan(plan):
    """PLAN_SPEC §5 invariants 1-4 on contributor *sets* per (rank, region) (:68 (i),(ii); Lemma 4 :340).

    Returns a dict of totals.  Raises PlanViolation on the first violated invariant."""
    p = plan.p
    fl = plan.flows
    region_len = {}
    holds = {}   # (rank, off) -> python int bitmask of contributors

    def get(rank, off):
        return holds.get((rank, off), 1 << rank)

    red = cop = 0
    for t in range(plan.n_steps):
        lo, hi = int(plan.step_begin[t]), int(plan.step_begin[t + 1])
        written, read = set(), set()
        for f in fl[lo:hi]:
            off, ln, src, dst = int(f["off"]), int(f["len"]), int(f["src"]), int(f["dst"])
            if int(f["step"]) != t:
                raise PlanViolation("step_begin does not index the step column")
            if region_len.setdefault(off, ln) != ln:
                raise PlanViolation(f"region at off {off} used with two lengths")
            if off + ln > plan.n or ln == 0 or src == dst:
                raise PlanViolation("bad range or self flow")
            if (dst, off) in written:
                raise PlanViolation(f"step {t}: two flows write ({dst},{off})")
            written.add((dst, off))
            read.add((src, off))
        if written & read:
            raise PlanViolation(f"step {t}: a flow reads a range written in the same step")
        # all flows of a step read the state before the step
        snapshot = {key: get(*key) for key in read}
        for f in fl[lo:hi]:
            off, ln, src, dst = int(f["off"]), int(f["len"]), int(f["src"]), int(f["dst"])
            s = snapshot[(src, off)]
            if f["op"] == P.REDUCE:
                d = get(dst, off)
                if s & d:
                    raise PlanViolation(f"step {t}: reduce joins overlapping contributor sets ({src}->{dst}, off {off})")
                holds[(dst, off)] = s | d
                red += ln
            else:
                holds[(dst, off)] = s
                cop += ln
    full = (1 << p) - 1
    # regions tile [0, n) exactly once
    offs = sorted(region_len)
    pos = 0
    for off in offs:
        if off != pos:
            raise PlanViolation(f"regions leave a gap or overlap at element {pos}")
        pos = off + region_len[off]
    if pos != plan.n:
        raise PlanViolation("regions do not cover [0, n)")
    for r in range(p):
        for off in offs:
            if get(r, off) != full:
                raise PlanViolation(f"rank {r} region {off}: contributors {get(r, off):b} != all ranks once")
    if red != (p - 1) * plan.n or cop != (p - 1) * plan.n:
        raise PlanViolation(f"traffic: reduce {red}, copy {cop}, expected {(p - 1) * plan.n} each (Lemma 4)")
    return {"reduce_elems": red, "copy_elems": cop, "n_regions": len(offs)}


def element_masks(plan):
    """Per-element contributor masks after the whole plan: uint64 array [p, n, W], W = ceil(p/64).

    Word w of rank r element e has bit i set iff rank 64*w+i contributed.  Also returns the number of
    elements at which a reduce saw overlapping sets (0 for a correct plan)."""
    p, n = plan.p, plan.n
    Wd = (p + 63) // 64
    m = np.zeros((p, n, Wd), dtype=np.uint64)
    for r in range(p):
        m[r, :, r // 64] = np.uint64(1) << np.uint64(r % 64)
    overlaps = 0
    for t in range(plan.n_steps):
        lo, hi = int(plan.step_begin[t]), int(plan.step_begin[t + 1])
        staged = []
        for f in plan.flows[lo:hi]:
            a, b = int(f["off"]), int(f["off"]) + int(f["len"])
            staged.append((f, m[int(f["src"]), a:b].copy()))
        for f, s in staged:
            a, b = int(f["off"]), int(f["off"]) + int(f["len"])
            d = m[int(f["dst"]), a:b]
            if f["op"] == P.REDUCE:
                overlaps += int(np.count_nonzero((s & d).any(axis=1)))
                m[int(f["dst"]), a:b] = s | d
            else:
                m[int(f["dst"]), a:b] = s
    return m, overlaps


def full_mask_words(p):
    """The all-ranks mask as W uint64 words."""
    Wd = (p + 63) // 64
    out = np.zeros(Wd, dtype=np.uint64)
    for r in range(p):
        out[r // 64] |= np.uint64(1) << np.uint64(r % 64)
    return out


def run_f32(plan, x):
    """Execute the plan on float32 arrays x[p, n]: each reduce flow is one IEEE fp32 add per element,
    each copy a bit copy, in table order (:126, :132, :136).  Returns the p outputs [p, n] float32."""
    y = np.array(x, dtype=np.float32, copy=True)
    assert y.shape == (plan.p, plan.n)
    for f in plan.flows:
        a, b = int(f["off"]), int(f["off"]) + int(f["len"])
        if f["op"] == P.REDUCE:
            y[int(f["dst"]), a:b] = y[int(f["dst"]), a:b] + y[int(f["src"]), a:b]
        else:
            y[int(f["dst"]), a:b] = y[int(f["src"]), a:b]
    return y


def bf16_bits_to_f32(b):
    """bf16 stored as uint16 -> float32 (exact)."""
    return (np.asarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def f32_to_bf16_bits(x):
    """float32 -> bf16 bits, round to nearest even (finite inputs; NaN kept quiet)."""
    u = np.asarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = (u + np.uint32(0x7FFF) + lsb) >> np.uint32(16)
    nan = (u & np.uint32(0x7FFFFFFF)) > np.uint32(0x7F800000)
    r = np.where(nan, (u >> np.uint32(16)) | np.uint32(0x40), r)
    return r.astype(np.uint16)


def run_bf16(plan, xb):
    """Execute the plan on bf16 data (uint16 bit patterns xb[p, n]) with fp32 partials and ONE final
    RNE rounding: a range's partial sum stays fp32 until a reduce completes the sum over
    all p ranks; that reduce rounds to bf16; copies move the stored value unchanged.
    Returns uint16 bits [p, n]."""
    p = plan.p
    val = bf16_bits_to_f32(xb).copy()          # current value of every (rank, element), fp32 carrier
    cnt = {}                                    # (rank, off) -> number of contributors held
    for f in plan.flows:
        a, b = int(f["off"]), int(f["off"]) + int(f["len"])
        s, d = int(f["src"]), int(f["dst"])
        cs, cd = cnt.get((s, a), 1), cnt.get((d, a), 1)
        if f["op"] == P.REDUCE:
            r = val[d, a:b] + val[s, a:b]
            if cs + cd == p:
                r = bf16_bits_to_f32(f32_to_bf16_bits(r))
            val[d, a:b] = r
            cnt[(d, a)] = cs + cd
        else:
            val[d, a:b] = val[s, a:b]
            cnt[(d, a)] = cs
    return f32_to_bf16_bits(val)    # exact: every final value is already a bf16 number


def run_f32_at(plan, x_cols, idx):
    """run_f32 restricted to the sampled element indices `idx` (sorted, unique): x_cols[p, len(idx)] holds the
    inputs at those elements.  Same walk, same one-IEEE-add-per-reduce-flow arithmetic, applied only to the
    samples a flow's range covers -- lets full-size runs be checked element by element on a sample."""
    idx = np.asarray(idx, dtype=np.int64)
    assert (np.diff(idx) > 0).all()
    y = np.array(x_cols, dtype=np.float32, copy=True)
    assert y.shape == (plan.p, len(idx))
    lo = np.searchsorted(idx, plan.flows["off"].astype(np.int64), side="left")
    hi = np.searchsorted(idx, (plan.flows["off"] + plan.flows["len"]).astype(np.int64), side="left")
    for f, a, b in zip(plan.flows, lo, hi):
        if a == b:
            continue
        if f["op"] == P.REDUCE:
            y[int(f["dst"]), a:b] = y[int(f["dst"]), a:b] + y[int(f["src"]), a:b]
        else:
            y[int(f["dst"]), a:b] = y[int(f["src"]), a:b]
    return y


def run_bf16_at(plan, xb_cols, idx):
    """run_bf16 restricted to sampled element indices (see run_f32_at): fp32 partials, one RNE rounding when a
    range's sum over all p ranks completes (R12).  xb_cols: uint16 bit patterns [p, len(idx)]."""
    idx = np.asarray(idx, dtype=np.int64)
    assert (np.diff(idx) > 0).all()
    p = plan.p
    val = bf16_bits_to_f32(xb_cols).copy()
    cnt = {}
    lo = np.searchsorted(idx, plan.flows["off"].astype(np.int64), side="left")
    hi = np.searchsorted(idx, (plan.flows["off"] + plan.flows["len"]).astype(np.int64), side="left")
    for f, a, b in zip(plan.flows, lo, hi):
        s, d, off = int(f["src"]), int(f["dst"]), int(f["off"])
        cs, cd = cnt.get((s, off), 1), cnt.get((d, off), 1)
        if f["op"] == P.REDUCE:
            if a != b:
                r = val[d, a:b] + val[s, a:b]
                if cs + cd == p:
                    r = bf16_bits_to_f32(f32_to_bf16_bits(r))
                val[d, a:b] = r
            cnt[(d, off)] = cs + cd
        else:
            if a != b:
                val[d, a:b] = val[s, a:b]
            cnt[(d, off)] = cs
    return f32_to_bf16_bits(val)
