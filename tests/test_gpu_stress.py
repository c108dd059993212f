"""Randomised stress of the dataflow executor's dependency protocol (pytest -m gpu): many small seeded plans with tiny
tiles and odd grids, so that tile-ops of different steps interleave as much as possible; every output must equal the
oracle's plan-order walk bit for bit and the verifier's masks must be complete."""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import interpreter as OI

pytestmark = pytest.mark.gpu


def _random_case(rng):
    kind = rng.integers(0, 5)
    if kind == 0:      # one straggler, bubble filling or not
        p = int(rng.integers(3, 25)); g = 1
        st = {int(rng.integers(0, p)): float(rng.choice([8 / 7, 4 / 3, 1.6, 2.0, 3.0]))}
    elif kind == 1:    # several stragglers
        p = int(rng.integers(5, 20)); g = 1
        m = int(rng.integers(2, min(4, p - 2) + 1))
        st = {int(r): float(rng.choice([8 / 7, 4 / 3, 2.0])) for r in rng.choice(p, size=m, replace=False)}
    elif kind == 2:    # multi-GPU servers, one straggler server
        g = int(rng.choice([2, 4])); q = int(rng.integers(3, 7)); p = g * q
        v = int(rng.integers(0, q)); l = float(rng.choice([8 / 7, 2.0]))
        st = {v * g + i: l for i in range(g)}
    elif kind == 3:    # no straggler: plain ring
        p = int(rng.integers(3, 20)); g = 1; st = {}
    else:              # ordering (1)
        p = int(rng.integers(3, 16)); g = 1
        st = {int(rng.integers(0, p)): float(rng.choice([1.5, 2.0, 3.0]))}
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    n = int(rng.integers(1, 60000))
    k = int(rng.choice([0, 4, 8]))
    dtype = int(rng.integers(0, 2))
    tile = int(rng.choice([1, 2, 7, 64, 224, 0]))
    grid = int(rng.choice([0, 0, 3, 37, 148]))
    return p, g, ell, n, k, dtype, tile, grid, (1 if kind == 4 else 0)


@pytest.mark.parametrize("seed", range(40))
def test_dataflow_random_plans(seed):
    from paper_2606_01680_b200.device import Session
    rng = np.random.default_rng(1000 + seed)
    p, g, ell, n, k, dtype, tile, grid, ordering = _random_case(rng)
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=B.OPTCC_EXEC_DATAFLOW, tile_units=tile, grid_ctas=grid, ordering=ordering)
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k, ordering=ordering or 2)
    w = W.Workload("stress", p, g, tuple(ell), n, dtype, "normal", 1.0, 5000 + seed)
    x = W.all_inputs(w)
    s = Session(plan, verify=(p <= 128))
    for _ in range(2):          # twice on the same session: counters and ticket must reset cleanly
        s.upload(x)
        s.execute()
        y = s.download()
        y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
        assert y.tobytes() == y_or.tobytes()
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0


@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_COLUMN])
@pytest.mark.parametrize("seed", range(16))
def test_dataflow_random_midsize_plans(seed, exec_mode):
    """Mid-size plans (sections of several thousand 16-byte units, odd tile sizes): the full streaming rounds, the
    partially entered last rounds, the remainder batches and the dead-source discard all occur; outputs bit-equal to
    the oracle, masks complete, and the per-step executor agrees on every element."""
    from paper_2606_01680_b200.device import Session
    rng = np.random.default_rng(7000 + seed)
    p = int(rng.integers(3, 10))
    st = {int(rng.integers(0, p)): float(rng.choice([8 / 7, 1.5, 2.0, 3.0]))}
    if seed % 4 == 3 and p >= 6:
        st[int((list(st)[0] + 2) % p)] = 4.0 / 3.0
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    dtype = int(rng.integers(0, 2))
    n = int(rng.integers(300_000, 1_500_000))
    k = int(rng.choice([4, 8]))
    tile = int(rng.choice([0, 1792, 3584, 1000, 5000, 3583]))
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, exec_mode=exec_mode, tile_units=tile)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k)
    w = W.Workload("mid", p, 1, tuple(ell), n, dtype, "normal", 1.0, 9000 + seed)
    x = W.all_inputs(w)
    s = Session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0
    assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()


@pytest.mark.parametrize("seed", list(range(150)) + [f"column-{i}" for i in range(80)])
def test_random_plans_any_executor_any_verifier(seed):
    """Random plans through a random executor, with the lazy or the eager verifier, complete or cut after a random
    step: outputs (complete schedules) bit-equal to the oracle; masks, number of wrong final masks, first wrong
    index and overlap count equal to the oracle's walk of the same (possibly truncated) table.  The "column-i" cases
    run the column executor (twice on the same session: its ticket must reset cleanly)."""
    import dataclasses
    from paper_2606_01680_b200.device import Session
    column = isinstance(seed, str)
    if column:
        seed = 500 + int(seed.split("-")[1])
    rng = np.random.default_rng(31337 + seed)
    p, g, ell, n, k, dtype, tile, grid, ordering = _random_case(rng)
    mode = int(rng.integers(1, 4))      # persistent, per-step or dataflow
    if column:
        mode = B.OPTCC_EXEC_COLUMN
    eager = int(rng.integers(0, 2))
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k, ordering=ordering or 2)
    limit = 0
    if rng.integers(0, 3) == 0 and oplan.n_steps > 2:
        limit = int(rng.integers(max(1, oplan.n_steps - 6), oplan.n_steps))
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=mode, tile_units=tile, grid_ctas=grid, ordering=ordering,
                        verify_eager=eager, step_limit=limit)
    if eager:
        assert plan.info["lazy_verify"] == 0
    elif not limit:
        assert plan.info["lazy_verify"] == 1
    s = Session(plan, verify=True)
    if not limit:
        x = W.all_inputs(W.Workload("s", p, g, tuple(ell), n, dtype, "normal", 1.0, 77000 + seed))
        y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
        for _ in range(2 if column else 1):
            s.upload(x)
            s.execute()
            assert s.download().tobytes() == y_or.tobytes()
    else:
        oplan = dataclasses.replace(oplan, n_steps=limit)
    res = s.verify(raise_on_fail=False)
    m_or, overlaps = OI.element_masks(oplan)
    assert s.masks().tobytes() == m_or.tobytes()
    bad = (m_or != OI.full_mask_words(p)[None, None, :]).any(axis=2)
    assert res["bad_elements"] == int(bad.sum())
    assert res["overlap_elements"] == overlaps
    if bad.any():
        assert res["first_bad"] == int(np.flatnonzero(bad.reshape(-1))[0])


_SOAK = int(__import__("os").environ.get("OPTCC_SOAK", "0"))      # extra seeds for a one-off soak run


@pytest.mark.parametrize("seed", range(60 + _SOAK))
def test_column_executor_random_cuts_leave_the_oracles_state(seed):
    """The column executor keeps partial sums in registers and does not store the ones a later EXECUTED flow overwrites
    (opts.no_forward = 0): whatever the plan, the tile size (one round or several, CTA- or warp-wide), the forwarding
    mode and the step the schedule is cut at, every element of every rank buffer must hold what the oracle holds after
    walking the same table prefix (fp32 plans: the rank buffers show every partial sum)."""
    import dataclasses
    from paper_2606_01680_b200.device import Session
    rng = np.random.default_rng(424242 + seed)
    p, g, ell, n, k, _, _, grid, ordering = _random_case(rng)
    n = int(rng.integers(1, 400000))
    tile = int(rng.choice([0, 0, 128, 64, 1792, 896, 3584, 224]))
    no_forward = int(rng.choice([0, 0, 0, 1, 2]))
    oplan = OP.build_plan(p, g, ell, n, W.F32, k=k, ordering=ordering or 2)
    limit = 0 if (oplan.n_steps < 2 or rng.integers(0, 4) == 0) else int(rng.integers(1, oplan.n_steps))
    plan = B.optcc_plan(p, g, ell, n, W.F32, k=k, exec_mode=B.OPTCC_EXEC_COLUMN, tile_units=tile, grid_ctas=grid,
                        ordering=ordering, step_limit=limit, no_forward=no_forward)
    x = W.all_inputs(W.Workload("cut", p, g, tuple(ell), n, W.F32, "normal", 1.0, 88000 + seed))
    s = Session(plan)
    s.upload(x)
    s.execute()
    y = s.download()
    if limit:
        oplan = dataclasses.replace(oplan, n_steps=limit, flows=oplan.flows[:int(oplan.step_begin[limit])],
                                    step_begin=oplan.step_begin[:limit + 1])
    assert y.tobytes() == OI.run_f32(oplan, x).tobytes(), (p, g, n, k, tile, no_forward, limit)
