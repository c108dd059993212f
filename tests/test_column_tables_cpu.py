"""The column executor's host tables, checked WITHOUT a GPU (optcc_column_tables): the region-by-region work list the
kernel runs -- chain-ordered lists, storage kinds, first-touch / last-write / dead-source flags and the bulk all-gather
flags -- is interpreted here in numpy exactly as the kernel interprets it and must reproduce the oracle's plan-order
walk bit for bit.  Dead sources are poisoned after their flow has read them and the staged tile replaces the source of
every DFLOW_FROM_STAGE copy, so a wrong flag or an order that breaks a data dependency shows up as a
wrong output."""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import interpreter as OI

DEAD_SRC, SRC_INIT, DST_INIT, FINAL, STAGE_OUT, FROM_STAGE, SRC_FWD, NO_STORE, SRC_REG = 1, 2, 4, 8, 64, 128, 256, 512, 1024


def _simulate(plan, x, bulk=True, fwd=False):
    """numpy interpretation of the records: returns the p outputs (f32 array or bf16 bit patterns).  fwd: also act on
    DFLOW_SRC_FWD / DFLOW_NO_STORE as the lazy contributor-mask run does (the source is what the previous flow
    produced, taken from registers; a result nobody reads from memory is not stored -- its range is poisoned here)."""
    info = plan.info
    rec, items = B.optcc_column_tables(plan)
    p, n = info["p"], info["n"]
    bf16 = info["dtype"] == B.OPTCC_BF16
    buf = OI.bf16_bits_to_f32(x).copy() if bf16 else np.array(x, dtype=np.float32, copy=True)   # rank buffers (value carrier)
    shadow = np.full((p, n), np.nan, dtype=np.float32)                                         # fp32 partials (bf16 plans)
    written = np.zeros((p, n), dtype=bool)
    # one list per region: the items of a region share [first, end)
    lists = sorted({(int(i["first"]), int(i["end"])) for i in items})
    assert sum(e - f for f, e in lists) == len(rec), "every record belongs to exactly one region's list"
    # the items tile every region: tiles 0..T-1 with tile_units units each, the last one shorter
    for first, end in lists:
        L = rec[first:end]
        off, ln = int(L[0]["off"]), int(L[0]["len"])
        assert (L["off"] == off).all() and (L["len"] == ln).all()
        a, b = off, off + ln
        stage = None
        prev = None
        final_seen = np.zeros(p, dtype=bool)
        for i, f in enumerate(L):
            s, d, fl = int(f["src"]), int(f["dst"]), int(f["flags"])
            if fl & SRC_FWD:
                assert i > 0 and int(L[i - 1]["dst"]) == s and f["op"] == 0 and not (int(L[i - 1]["flags"]) & FROM_STAGE)
            if fl & NO_STORE:
                assert i + 1 < len(L) and (int(L[i + 1]["flags"]) & SRC_FWD) and not (fl & (FINAL | STAGE_OUT | FROM_STAGE))
            assert bool(fl & SRC_INIT) == (not written[s, a]), "SRC_INIT = no earlier flow wrote the source range"
            assert bool(fl & DST_INIT) == (not written[d, a]), "DST_INIT = no earlier flow wrote the destination range"
            assert not final_seen[d], "a flow writes a range after its DFLOW_FINAL write"
            src = shadow[s, a:b] if (bf16 and f["ksrc"]) else buf[s, a:b]
            if fwd and (fl & SRC_FWD):
                src = prev
            if fl & SRC_REG:   # data runs: the registers the previous (reduce) flow stored are this flow's source operand
                assert i > 0 and f["op"] == 0 and L[i - 1]["op"] == 0 and int(L[i - 1]["dst"]) == s
                assert not bf16 or int(L[i - 1]["kdout"]) == int(f["ksrc"])
                if not fwd:
                    assert src.tobytes() == prev.tobytes()     # memory holds the same bits: the store was issued
                src = prev
            if f["op"] == 0:
                din = shadow[d, a:b] if (bf16 and f["kdin"]) else buf[d, a:b]
                r = din + src
                if bf16 and not f["kdout"]:
                    r = OI.bf16_bits_to_f32(OI.f32_to_bf16_bits(r))
                assert not (fl & FROM_STAGE)
                if fl & STAGE_OUT:
                    assert bulk and not (bf16 and f["kdout"])
                    stage = r.copy()
            else:
                assert not (fl & (STAGE_OUT | DEAD_SRC))
                if fl & FROM_STAGE:
                    assert bulk and stage is not None and not (bf16 and (f["ksrc"] or f["kdout"]))
                    r = stage                      # the copy's source is never read: the staged tile is stored
                else:
                    r = src.copy()
            prev = np.array(r, copy=True)
            if fwd and (fl & NO_STORE):
                r = np.full_like(r, np.nan)
            if bf16 and f["kdout"]:
                shadow[d, a:b] = r
            else:
                buf[d, a:b] = r
            written[d, a:b] = True
            if fl & FINAL:
                final_seen[d] = True
            if fl & DEAD_SRC:                      # the lines are dropped from the caches: nobody may read them again
                (shadow if (bf16 and f["ksrc"]) else buf)[s, a:b] = np.nan
    return OI.f32_to_bf16_bits(buf) if bf16 else buf, items, lists


CASES = [
    # p, g, stragglers, n, dtype, k, extra options
    (4, 1, {0: 2.0}, 4099, W.F32, 8, {}),
    (5, 1, {2: 1.5}, 50001, W.F32, 4, {}),                                   # bubble filling
    (16, 1, {0: 8.0 / 7.0}, 2 ** 14 + 2, W.F32, 8, {}),                      # C2 shape
    (6, 1, {}, 7777, W.F32, 0, {}),                                          # plain ring
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 6553, W.F32, 4, {}),                      # several stragglers
    (16, 4, {r: 2.0 for r in range(4)}, 40001, W.F32, 4, {}),                # g > 1: collect / NIC / distribute chains
    (32, 8, {r: 2.0 for r in range(8)}, 30011, W.F32, 8, {}),                # C4 shape, scaled down
    (24, 4, {0: 1.5, 1: 1.5, 2: 1.5, 3: 1.5, 8: 3.0, 9: 3.0, 10: 3.0, 11: 3.0}, 9001, W.F32, 4, {}),   # two straggler servers
    (9, 1, {4: 3.0}, 12345, W.F32, 4, {"ordering": 1}),
    (9, 1, {4: 3.0}, 12345, W.F32, 8, {"ordering": 3}),                      # the four-pattern mix
    (16, 1, {0: 8.0 / 7.0}, 2 ** 14 + 2, W.BF16, 8, {"ordering": 3}),
    (16, 1, {3: 4.0 / 3.0}, 20001, W.F32, 0, {"schedule": 1}),               # ring on the degraded topology
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 70001, W.BF16, 4, {}),   # C3 shape, bf16 with fp32 partials
    (5, 1, {2: 1.5}, 50003, W.BF16, 4, {}),
    (12, 2, {0: 1.5, 1: 1.5}, 4097, W.BF16, 12, {}),
    (3, 1, {1: 3.0}, 5, W.F32, 4, {}),                                       # most flows dropped
    (16, 1, {0: 8.0 / 7.0}, 2 ** 14 + 2, W.F32, 8, {"col_order": 1}),        # table order
    (16, 4, {r: 2.0 for r in range(4)}, 40001, W.F32, 4, {"copy_path": 1}),  # no bulk all-gather path
    (16, 4, {r: 2.0 for r in range(4)}, 40001, W.F32, 4, {"no_discard": 1}),
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_column_tables_reproduce_the_oracle(case):
    p, g, st, n, dtype, k, extra = CASES[case]
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=B.OPTCC_EXEC_COLUMN, **extra)
    okw = {key: extra[key] for key in ("ordering", "schedule") if key in extra}
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k, **okw)
    x = W.all_inputs(W.Workload("t", p, g, tuple(ell), n, dtype, "normal", 1.0, 300 + case))
    y, items, lists = _simulate(plan, x, bulk=extra.get("copy_path", 0) != 1)
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    # the forwarding flags as the default data run (opts.no_forward = 0) and the lazy verifier act on them: a partial sum
    # with DFLOW_NO_STORE is never stored (its range is poisoned here), the flow after it takes it from registers
    y2, _, _ = _simulate(plan, x, bulk=extra.get("copy_path", 0) != 1, fwd=True)
    assert y2.tobytes() == y_or.tobytes()
    rec, _ = B.optcc_column_tables(plan)
    if extra.get("copy_path", 0) == 1:
        assert not (rec["flags"] & (STAGE_OUT | FROM_STAGE)).any()
    else:   # every all-gather copy of an AllReduce plan goes through the stage
        assert ((rec["flags"][rec["op"] == 1] & FROM_STAGE) != 0).all()
    if extra.get("no_discard", 0):
        assert not (rec["flags"] & DEAD_SRC).any()
    # the work items tile every region exactly once
    A = plan.info["unit_elems"]
    by_list = {}
    for it in items:
        by_list.setdefault((int(it["first"]), int(it["end"])), []).append((int(it["tile"]), int(it["units"])))
    for (first, end), tiles in by_list.items():
        tiles.sort()
        units = -(-int(rec[first]["len"]) // A)
        assert [t for t, _ in tiles] == list(range(len(tiles))) and sum(u for _, u in tiles) == units


@pytest.mark.parametrize("case", [1, 2, 5, 6, 10, 13])
@pytest.mark.parametrize("frac", [0.3, 0.7])
def test_column_tables_of_a_truncated_schedule(case, frac):
    """step_limit: the lists hold the flows of the executed steps only (general path, no class replication) and
    reproduce the oracle's walk of the table prefix; nothing is marked dead (the overwrite might never run)."""
    import dataclasses
    p, g, st, n, dtype, k, extra = CASES[case]
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k, **{key: extra[key] for key in ("ordering", "schedule") if key in extra})
    limit = max(1, int(oplan.n_steps * frac))
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=B.OPTCC_EXEC_COLUMN, step_limit=limit, **extra)
    x = W.all_inputs(W.Workload("t", p, g, tuple(ell), n, dtype, "normal", 1.0, 500 + case))
    y, _, _ = _simulate(plan, x, fwd=True)    # as the default data run: unstored partial sums are poisoned
    rec, _ = B.optcc_column_tables(plan)
    assert not (rec["flags"] & DEAD_SRC).any()
    prefix = dataclasses.replace(oplan, n_steps=limit, flows=oplan.flows[:int(oplan.step_begin[limit])],
                                 step_begin=oplan.step_begin[:limit + 1])
    if dtype == W.F32:
        assert y.tobytes() == OI.run_f32(prefix, x).tobytes()
    # (bf16 prefixes leave partial sums in the fp32 partials, which the rank buffers do not show: f32 cases only)


def test_chain_order_keeps_collect_chains_together():
    """C4's shape: in table order the collect hops of the q servers interleave; in the executor's order a flow is
    followed by the flow that reads what it wrote, so each server's chain is contiguous."""
    p, g = 32, 8
    ell = [2.0] * 8 + [1.0] * 24
    plan = B.optcc_plan(p, g, ell, 30011, W.F32, k=8, exec_mode=B.OPTCC_EXEC_COLUMN)
    rec, items = B.optcc_column_tables(plan)
    first, end = int(items[0]["first"]), int(items[0]["end"])
    L = rec[first:end]
    follows = sum(1 for i in range(1, len(L)) if L[i]["src"] == L[i - 1]["dst"] or L[i]["dst"] == L[i - 1]["dst"])
    plan_t = B.optcc_plan(p, g, ell, 30011, W.F32, k=8, exec_mode=B.OPTCC_EXEC_COLUMN, col_order=1)
    rec_t, items_t = B.optcc_column_tables(plan_t)
    Lt = rec_t[int(items_t[0]["first"]):int(items_t[0]["end"])]
    follows_t = sum(1 for i in range(1, len(Lt)) if Lt[i]["src"] == Lt[i - 1]["dst"] or Lt[i]["dst"] == Lt[i - 1]["dst"])
    assert follows > 0.8 * (len(L) - 1) > follows_t


def test_auto_executor_is_reported():
    """OPTCC_EXEC_AUTO (the default of optcc_plan) resolves to the column executor on the five config shapes."""
    for ci in range(5):
        w = W.config(ci).scaled(2 ** 14)
        plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype)
        assert plan.info["exec_mode"] == B.OPTCC_EXEC_COLUMN
        rec, items = B.optcc_column_tables(plan)
        assert len(rec) == plan.info["n_flows"] and len(items) > 0
    plan = B.optcc_plan(4, 1, [2.0, 1.0, 1.0, 1.0], 4096, W.F32, exec_mode=B.OPTCC_EXEC_DATAFLOW)
    assert plan.info["exec_mode"] == B.OPTCC_EXEC_DATAFLOW
    with pytest.raises(B.OptccError):
        B.optcc_column_tables(plan)


def test_ring_hops_take_their_source_from_registers():
    """DFLOW_SRC_REG: in a chain-ordered list every reduce hop after the first follows the flow that stored its source
    (plain ring: p - 1 reduce flows per region, p - 2 of them flagged); in table order with k > 1 nothing changes for a
    ring either (one chain per region), and copies are never flagged."""
    p, n = 6, 7777
    plan = B.optcc_plan(p, 1, [1.0] * p, n, W.F32, k=0, exec_mode=B.OPTCC_EXEC_COLUMN)
    rec, items = B.optcc_column_tables(plan)
    lists = sorted({(int(i["first"]), int(i["end"])) for i in items})
    for first, end in lists:
        L = rec[first:end]
        red = L[L["op"] == 0]
        assert len(red) == p - 1 and int(((red["flags"] & SRC_REG) != 0).sum()) == p - 2
        assert not (L["flags"][L["op"] == 1] & SRC_REG).any()
