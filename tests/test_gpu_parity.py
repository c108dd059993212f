"""GPU parity tests (run on the B200 box: pytest -m gpu).  Every call goes through the C-ABI (binding -> liboptcc).

Bars (BASELINE.json north_star):
  * contributor masks equal the oracle's element by element, bit-exactly; plan tables too (CPU test file);
  * fp32 outputs: |y - y_ref| <= p 2^-23 sum_i |x_i| per element against the fp64 reference sum, AND bit-identical
    to the oracle's plan-order fp32 emulation (each reduce flow is one IEEE add per element in a plan-fixed order);
  * bf16 outputs: within 2^-7 relative (+ fp32 accumulation floor, R12) of the fp64 reference, AND bit-identical to
    the oracle's fp32-partials / one-final-RNE emulation;
  * all p outputs bitwise identical (PAPER.md:68 (ii)).
"""
import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import workloads as W
from oracle import planner as OP
from oracle import interpreter as OI
from oracle import reference as OR

pytestmark = pytest.mark.gpu

MODES = [B.OPTCC_EXEC_PERSISTENT, B.OPTCC_EXEC_PER_STEP, B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_COLUMN]


def _session(plan, verify=False):
    from paper_2606_01680_b200.device import Session
    return Session(plan, verify=verify)


def _wl(p, g, st, n, dtype, seed, dist="normal"):
    ell = tuple(float(st.get(i, 1.0)) for i in range(p))
    return W.Workload(f"t{p}x{n}", p, g, ell, n, dtype, dist, 1.0, seed)


def _run_and_check(w, k, exec_mode, grid_ctas=0, **opts):
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=exec_mode, grid_ctas=grid_ctas, **opts)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    x = W.all_inputs(w)
    s = _session(plan)
    s.upload(x)
    s.execute()
    y = s.download()
    assert OR.all_ranks_identical(y)
    if w.dtype == W.F32:
        assert OR.check_f32(y[0], x).all()                       # north_star fp32 bound vs the fp64 sum
        y_or = OI.run_f32(oplan, x)
        assert y.view(np.uint32).tobytes() == y_or.view(np.uint32).tobytes()   # plan-order bit parity
    else:
        xf = OI.bf16_bits_to_f32(x)
        assert OR.check_bf16(OI.bf16_bits_to_f32(y[0]), xf).all()
        y_or = OI.run_bf16(oplan, x)
        assert y.tobytes() == y_or.tobytes()
    return plan, s


# sizes: a few hundred KB per rank so that slices, unrolled bodies, remainders and ragged tails are all exercised
F32_CASES = [
    # p, g, stragglers, n, k
    (4, 1, {0: 2.0}, 2 ** 16, 8),                       # C1 shape, scaled n
    (4, 1, {0: 2.0}, 100003, 4),                        # ragged: n % 4 = 3
    (5, 1, {2: 1.5}, 50001, 4),                         # bubble filling (l < 2), ragged n % 4 = 1
    (16, 1, {0: 8.0 / 7.0}, 2 ** 17 + 2, 8),            # C2 shape
    (6, 1, {}, 77777, 0),                               # C0 plain ring
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 65539, 4),           # C2 construction, m = 2
    (16, 4, {r: 2.0 for r in range(4)}, 40001, 4),      # C3 construction, g = 4
    (32, 1, {0: 2.0 - 1.0 / 31.0}, 2 ** 15, 12),        # C5 shape at the Thm-1 switch
    (3, 1, {1: 3.0}, 5, 4),                             # fewer units than sections: most flows dropped
    (3, 1, {0: 2.0}, 1, 4),                             # one element
]


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("p,g,st,n,k", F32_CASES)
def test_f32_parity(p, g, st, n, k, exec_mode):
    _run_and_check(_wl(p, g, st, n, W.F32, seed=100 + p), k, exec_mode)


BF16_CASES = [
    (4, 1, {0: 2.0}, 2 ** 16, 8),
    (5, 1, {2: 1.5}, 50003, 4),                         # ragged: n % 8 = 3
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 70001, 4),   # C3 shape (config 3), ragged
    (6, 1, {}, 33333, 0),
    (12, 2, {0: 1.5, 1: 1.5}, 4097, 12),
    (3, 1, {0: 2.0}, 1, 4),
]


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("p,g,st,n,k", BF16_CASES)
def test_bf16_parity(p, g, st, n, k, exec_mode):
    _run_and_check(_wl(p, g, st, n, W.BF16, seed=200 + p), k, exec_mode)


# Column executor, opts.no_forward: 0 = partial sums travel between consecutive flows of a column in registers and a
# partial sum nobody else reads is not stored; 1 = every flow loads both operands and stores its result; 2 = registers
# are forwarded, every result is stored.  Tile sizes: CTA-wide one-round tiles (1792 units f32 / 896 bf16), warp-wide
# tiles (128), and tiles of more than one round (3584: the forwarding instantiation is not used).
FWD_CASES = [
    # p, g, stragglers, n, dtype, k, tile_units
    (16, 1, {0: 8.0 / 7.0}, 2 ** 21 + 6, W.F32, 4, 0),        # C2 shape: regions of several CTA-wide tiles + a short one
    (16, 1, {0: 8.0 / 7.0}, 2 ** 17 + 2, W.F32, 8, 0),        # warp-wide tiles
    (5, 1, {2: 1.5}, 500001, W.F32, 4, 1792),                 # bubble filling, ragged end inside a CTA-wide tile
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 655390, W.F32, 4, 3584),   # two rounds per tile
    (16, 4, {r: 2.0 for r in range(4)}, 400001, W.F32, 4, 0), # g > 1: collect / NIC / distribute chains
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 2 ** 20 + 24, W.BF16, 4, 0),   # C3 shape, fp32 partials, warp-wide
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 2 ** 20 + 24, W.BF16, 4, 896), # CTA-wide
    (5, 1, {2: 1.5}, 500003, W.BF16, 4, 0),
    (12, 2, {0: 1.5, 1: 1.5}, 409700, W.BF16, 12, 1792),      # bf16 tiles of two rounds
]


@pytest.mark.parametrize("no_forward", [0, 1, 2])
@pytest.mark.parametrize("case", range(len(FWD_CASES)))
def test_column_executor_forwarding_modes_give_the_oracle_bits(case, no_forward):
    p, g, st, n, dtype, k, tile = FWD_CASES[case]
    _run_and_check(_wl(p, g, st, n, dtype, seed=700 + case), k, B.OPTCC_EXEC_COLUMN, tile_units=tile, no_forward=no_forward)


@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_PERSISTENT, B.OPTCC_EXEC_DATAFLOW])
@pytest.mark.parametrize("grid_ctas", [1, 7, 148])
def test_f32_parity_any_grid(grid_ctas, exec_mode):
    """Work is cut per CTA (slices) or claimed dynamically (tile-ops): the result must not depend on the grid."""
    _run_and_check(_wl(16, 1, {3: 4.0 / 3.0}, 2 ** 16 + 13, W.F32, seed=7), 8, exec_mode, grid_ctas)


BULK_CASES = [
    (4, 1, {0: 2.0}, 100003, W.F32, 4),                 # ragged n % 4 = 3: < 16-byte tail after the bulk part
    (16, 1, {0: 8.0 / 7.0}, 2 ** 18 + 2, W.F32, 8),     # bubble flows, tiles larger than one bulk round
    (5, 1, {2: 1.5}, 50003, W.BF16, 4),                 # bf16, ragged n % 8 = 3
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 70001, W.BF16, 4),
    (16, 4, {r: 2.0 for r in range(4)}, 40001, W.F32, 4),
    (3, 1, {0: 2.0}, 1, W.F32, 4),
]


@pytest.mark.parametrize("p,g,st,n,dtype,k", BULK_CASES)
def test_bulk_copy_path_parity(p, g, st, n, dtype, k):
    """copy_path = 2: the all-gather (copy) tile-ops are moved by cp.async.bulk (TMA 1-D bulk copies) instead of
    LDG/STG; outputs and masks must not change by a bit."""
    w = _wl(p, g, st, n, dtype, seed=300 + p)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=B.OPTCC_EXEC_DATAFLOW, copy_path=2)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    x = W.all_inputs(w)
    s = _session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0
    assert s.masks().tobytes() == OI.element_masks(oplan)[0].tobytes()


@pytest.mark.parametrize("tile_units", [1, 64, 4096])
def test_dataflow_parity_any_tile_size(tile_units):
    w = _wl(7, 1, {0: 2.0, 1: 4.0 / 3.0}, 20011, W.F32, seed=11)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4, exec_mode=B.OPTCC_EXEC_DATAFLOW, tile_units=tile_units)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=4)
    x = W.all_inputs(w)
    s = _session(plan)
    s.upload(x)
    s.execute()
    y = s.download()
    assert y.tobytes() == OI.run_f32(oplan, x).tobytes()


MASK_CASES = [
    (4, 1, {0: 2.0}, 4099, W.F32, 8), (5, 1, {2: 1.5}, 50001, W.F32, 4), (6, 1, {}, 7777, W.F32, 0),
    (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 9001, W.BF16, 4),
    (128, 8, {r: 2.0 for r in range(8)}, 6007, W.F32, 4),               # two mask words (p = 128)
    (72, 1, {1: 2.0}, 3001, W.BF16, 4),                                   # two mask words, p not a multiple of 64
    (16, 4, {r: 2.0 for r in range(4)}, 40001, W.F32, 4),
]


@pytest.mark.parametrize("eager", [0, 1])
@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("p,g,st,n,dtype,k", MASK_CASES)
def test_verifier_masks_equal_oracle(p, g, st, n, dtype, k, exec_mode, eager):
    """eager = 0: the lazy verifier (initial masks as constants, final masks checked by their last writer);
    eager = 1: the mask arrays are initialised and checked by separate passes.  Same masks, same verdict."""
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    plan = B.optcc_plan(p, g, ell, n, dtype, k=k, exec_mode=exec_mode, verify_eager=eager)
    assert plan.info["lazy_verify"] == 1 - eager          # a complete schedule writes every (rank, section)
    oplan = OP.build_plan(p, g, ell, n, dtype, k=k)
    s = _session(plan, verify=True)
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0
    assert res["checked"] == p * n and res["first_bad"] == 2 ** 64 - 1
    m_or, overlaps = OI.element_masks(oplan)
    assert overlaps == 0
    m = s.masks()
    assert m.shape == m_or.shape and m.tobytes() == m_or.tobytes()
    assert (m == OI.full_mask_words(p)[None, None, :]).all()


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("limit", [1, 9, 19])
def test_verifier_detects_a_truncated_schedule(limit, exec_mode):
    """The verifier is not vacuous: a schedule cut after `limit` steps must fail, with exactly the masks and
    the number of wrong elements the oracle's interpreter finds for the same truncated table."""
    import dataclasses
    p, n, k = 5, 4099, 4
    ell = [1.0, 1.0, 1.5, 1.0, 1.0]
    plan = B.optcc_plan(p, 1, ell, n, W.F32, k=k, exec_mode=exec_mode, step_limit=limit)
    oplan = OP.build_plan(p, 1, ell, n, W.F32, k=k)
    assert limit < oplan.n_steps
    s = _session(plan, verify=True)
    res = s.verify(raise_on_fail=False)
    m_or, _ = OI.element_masks(dataclasses.replace(oplan, n_steps=limit))
    m = s.masks()
    assert m.tobytes() == m_or.tobytes()
    bad = (m_or != OI.full_mask_words(p)[None, None, :]).any(axis=2)
    assert res["bad_elements"] == int(bad.sum()) > 0
    assert res["first_bad"] == int(np.flatnonzero(bad.reshape(-1))[0])
    with pytest.raises(B.OptccError) as e:
        s.verify()
    assert e.value.name == "EVERIFY"


LAZY_TRUNCATED = [
    # p, ell, k, ordering, schedule, limits that still write every (rank, section) -- so the lazy verifier runs
    (5, [1.0] * 5, 0, 0, 0, (5, 7)),                                   # C0: 8 steps, cut inside the all-gather
    (5, [1.0, 1.0, 1.5, 1.0, 1.0], 4, 1, 0, (24, 27)),                 # C1' (ordering 1): 28 steps
    (5, [1.0, 1.0, 2.5, 1.0, 1.0], 0, 0, 1, (6,)),                     # ring on the degraded topology
]


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("n", [4099, 150001])
@pytest.mark.parametrize("p,ell,k,ordering,schedule,limits", LAZY_TRUNCATED)
def test_lazy_verifier_detects_a_truncated_schedule(p, ell, k, ordering, schedule, limits, n, exec_mode):
    """Truncated schedules that still write every (rank, section) at least once are verified lazily: the wrong final
    masks are found by the last writer of each range (no pass over the arrays).  Count, first index and the masks
    themselves must equal the oracle's for the same truncated table -- and the eager verifier's."""
    import dataclasses
    oplan = OP.build_plan(p, 1, ell, n, W.F32, k=k, ordering=ordering or 2, schedule=schedule)
    for limit in limits:
        assert limit < oplan.n_steps
        m_or, _ = OI.element_masks(dataclasses.replace(oplan, n_steps=limit))
        bad = (m_or != OI.full_mask_words(p)[None, None, :]).any(axis=2)
        assert bad.sum() > 0
        for eager in (0, 1):
            plan = B.optcc_plan(p, 1, ell, n, W.F32, k=k, exec_mode=exec_mode, step_limit=limit, ordering=ordering,
                                schedule=schedule, verify_eager=eager)
            assert plan.info["lazy_verify"] == 1 - eager
            s = _session(plan, verify=True)
            res = s.verify(raise_on_fail=False)
            assert s.masks().tobytes() == m_or.tobytes()
            assert res["bad_elements"] == int(bad.sum())
            assert res["first_bad"] == int(np.flatnonzero(bad.reshape(-1))[0])
            assert res["overlap_elements"] == 0


def test_execute_rejects_bad_arguments():
    import torch
    plan = B.optcc_plan(4, 1, [2.0, 1.0, 1.0, 1.0], 4096, W.F32, k=4)
    s = _session(plan)
    bufs = list(s.bufs)
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute(plan, [bufs[0].data_ptr() + 4] + bufs[1:], s.ws_ptr, torch.cuda.current_stream().cuda_stream)
    assert e.value.name == "EINVAL"               # misaligned rank buffer
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute(plan, [0] + bufs[1:], s.ws_ptr, torch.cuda.current_stream().cuda_stream)
    assert e.value.name == "EINVAL"


def test_execute_host_roundtrip():
    import torch
    w = _wl(8, 1, {0: 2.0}, 2 ** 15 + 5, W.F32, seed=31)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4)
    s = _session(plan)
    x = W.all_inputs(w)
    hin = [torch.from_numpy(x[r].copy()).pin_memory() for r in range(w.p)]
    hout = [torch.empty(w.n, dtype=torch.float32).pin_memory() for r in range(w.p)]
    s.execute_host(hin, hout)
    torch.cuda.synchronize()
    y = np.stack([t.numpy() for t in hout])
    assert OR.all_ranks_identical(y)
    assert OR.check_f32(y[0], x).all()
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=4)
    assert y.tobytes() == OI.run_f32(oplan, x).tobytes()


@pytest.mark.parametrize("p,st,n,dtype,k,shards", [
    (8, {0: 2.0}, 2 ** 15 + 8, W.F32, 4, 3),
    (16, {0: 8.0 / 7.0}, 2 ** 18, W.F32, 8, 5),          # several tiles per flow, bubble flows
    (5, {2: 1.5}, 50000, W.BF16, 4, 4),
    (7, {0: 2.0, 1: 4.0 / 3.0}, 20011, W.F32, 4, 1),     # one shard: any n
    (130, {0: 2.0}, 1024, W.F32, 4, 2),                  # p > 128: the rank-pointer table is rewritten per shard
])
@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_COLUMN])
def test_execute_host_sharded_equals_the_oracle_shard_by_shard(p, st, n, dtype, k, shards, exec_mode):
    """optcc_execute_host_sharded: n_total = shards * n elements per rank, every shard an independent AllReduce with
    the one plan for n; the H2D / execute / D2H pipeline must give, shard by shard, exactly the oracle's plan-order
    result, and later work on the caller's stream must see the finished results."""
    import torch
    w = _wl(p, 1, st, n * shards, dtype, seed=77 + p)
    ell = list(w.ell)
    plan = B.optcc_plan(p, 1, ell, n, dtype, k=k, exec_mode=exec_mode)
    oplan = OP.build_plan(p, 1, ell, n, dtype, k=k)
    from paper_2606_01680_b200.device import Session
    s = Session(plan, shards=shards)
    x = W.all_inputs(w)                                   # [p, shards * n]
    tdt = torch.float32 if dtype == W.F32 else torch.int16
    hin = [torch.from_numpy(x[r].copy().view(np.float32 if dtype == W.F32 else np.int16)).pin_memory() for r in range(p)]
    hout = [torch.zeros(n * shards, dtype=tdt).pin_memory() for r in range(p)]
    for rep in range(2):                                  # the second call reuses the streams and events
        s.execute_host_sharded(hin, hout)
        on_stream = s.bufs[p - 1].clone()                 # enqueued on the caller's stream after the call
        torch.cuda.synchronize()
        y = np.stack([t.numpy().view(x.dtype) for t in hout])
        assert OR.all_ranks_identical(y)
        assert on_stream.cpu().numpy().view(x.dtype).tobytes() == y[0].tobytes() if dtype == W.F32 else True
        for c in range(shards):
            xs = np.ascontiguousarray(x[:, c * n:(c + 1) * n])
            y_or = OI.run_f32(oplan, xs) if dtype == W.F32 else OI.run_bf16(oplan, xs)
            assert np.ascontiguousarray(y[:, c * n:(c + 1) * n]).tobytes() == y_or.tobytes(), (rep, c)


def test_execute_host_sharded_rejects_bad_shapes():
    import torch
    plan = B.optcc_plan(4, 1, [2.0, 1.0, 1.0, 1.0], 4100, W.F32, k=4)     # n % 8 = 4
    from paper_2606_01680_b200.device import Session
    s = Session(plan, shards=2)
    h = [torch.zeros(8200).pin_memory() for _ in range(4)]
    st = torch.cuda.current_stream().cuda_stream
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute_host_sharded(plan, 8200, h, h, s.bufs, s.ws_ptr, st)    # shard start not 16-byte aligned
    assert e.value.name == "EINVAL"
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute_host_sharded(plan, 4101, h, h, s.bufs, s.ws_ptr, st)    # not a multiple of the plan's n
    assert e.value.name == "EINVAL"
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute_host_sharded(plan, 0, h, h, s.bufs, s.ws_ptr, st)
    assert e.value.name == "EINVAL"


@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_DATAFLOW, B.OPTCC_EXEC_COLUMN])
def test_execute_is_capturable_in_a_cuda_graph(exec_mode):
    """optcc_execute only enqueues work (two memsets and one cooperative launch once the tables are resident): it can
    be captured into a CUDA graph and replayed; every replay must reproduce the oracle's result."""
    import torch
    w = _wl(8, 1, {0: 2.0}, 2 ** 16 + 4, W.F32, seed=41)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4, exec_mode=exec_mode)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=4)
    x = W.all_inputs(w)
    y_or = OI.run_f32(oplan, x)
    s = _session(plan)
    s.upload(x)
    s.execute()                                    # warm-up: tables uploaded, kernel attributes set
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        s.execute(stream=side)
    for _ in range(3):
        s.upload(x)
        graph.replay()
        torch.cuda.synchronize()
        assert s.download().tobytes() == y_or.tobytes()


def test_repeated_execute_on_same_session_is_deterministic():
    w = _wl(16, 1, {0: 8.0 / 7.0}, 2 ** 16, W.F32, seed=5)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=8)
    s = _session(plan)
    x = W.all_inputs(w)
    outs = []
    for _ in range(3):
        s.upload(x)
        s.execute()
        outs.append(s.download([0, w.p - 1]).tobytes())
    assert outs[0] == outs[1] == outs[2]


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("dtype,n", [(W.F32, 100003), (W.BF16, 50003)])
def test_no_write_outside_the_rank_buffers(dtype, n, exec_mode):
    """compute-sanitizer is closed on this pool, so out-of-bounds writes are caught with guard bands: every rank
    buffer sits between two 4 KB canaries inside one allocation; after execute (ragged n, every executor) the
    canaries and the slack after element n-1 must be untouched and the result still bit-equal to the oracle."""
    import torch
    p, k = 6, 4
    w = _wl(p, 1, {2: 1.5}, n, dtype, seed=41)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=exec_mode)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    esz = 4 if dtype == W.F32 else 2
    guard = 4096
    stride = ((n * esz + 255) // 256) * 256 + 2 * guard
    from paper_2606_01680_b200.device import Session
    s = Session(plan, alloc_bufs=False)
    arena = torch.full((p * stride,), 0xA5, dtype=torch.uint8, device=s.device)
    base = arena.data_ptr()
    assert base % 256 == 0
    x = W.all_inputs(w)
    ptrs = []
    for r in range(p):
        off = r * stride + guard
        arena[off:off + n * esz] = torch.from_numpy(x[r].view(np.uint8).copy()).to(s.device)
        ptrs.append(base + off)
    B.optcc_execute(plan, ptrs, s.ws_ptr, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    host = arena.cpu().numpy()
    y = np.stack([host[r * stride + guard: r * stride + guard + n * esz].view(x.dtype) for r in range(p)])
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    for r in range(p):
        lo, hi = r * stride, r * stride + guard + n * esz
        assert (host[lo:lo + guard] == 0xA5).all(), f"rank {r}: write before the buffer"
        assert (host[hi:(r + 1) * stride] == 0xA5).all(), f"rank {r}: write past element n-1"


@pytest.mark.parametrize("exec_mode", MODES)
def test_more_than_128_ranks_use_the_pointer_table(exec_mode):
    """p > 128: rank pointers no longer fit the kernel parameters and travel through the workspace; contributor
    masks are limited to p <= 128 (R17), so optcc_verify must refuse with EUNSUPPORTED."""
    p, n, k = 160, 20001, 4
    w = _wl(p, 1, {7: 2.0}, n, W.F32, seed=160)
    plan, s = _run_and_check(w, k, exec_mode)
    assert plan.info["mask_words"] == 0
    with pytest.raises(B.OptccError) as e:
        s.verify()
    assert e.value.name == "EUNSUPPORTED"


def test_two_plans_alternate_on_one_workspace():
    """The workspace holds one plan's tables at a time; execute must notice that another plan used it in between."""
    import torch
    from paper_2606_01680_b200.device import Session
    wa = _wl(8, 1, {0: 2.0}, 40001, W.F32, seed=1)
    wb = _wl(8, 1, {3: 1.5}, 40001, W.F32, seed=2)
    pa = B.optcc_plan(wa.p, 1, wa.ell, wa.n, wa.dtype, k=4)
    pb = B.optcc_plan(wb.p, 1, wb.ell, wb.n, wb.dtype, k=8)
    sa = Session(pa)
    big = max(pa.info["workspace_bytes"], pb.info["workspace_bytes"])
    ws = torch.empty(int(big) + 256, dtype=torch.uint8, device=sa.device)
    ptr = ws.data_ptr() + (-ws.data_ptr()) % 256
    stream = torch.cuda.current_stream().cuda_stream
    for plan, w in ((pa, wa), (pb, wb), (pa, wa), (pb, wb)):
        x = W.all_inputs(w)
        sa.upload(x)
        B.optcc_execute(plan, sa.bufs, ptr, stream)
        y = sa.download()
        oplan = OP.build_plan(w.p, 1, list(w.ell), w.n, w.dtype, k=plan.info["k"])
        assert y.tobytes() == OI.run_f32(oplan, x).tobytes()


@pytest.mark.parametrize("dtype", [W.F32, W.BF16])
@pytest.mark.parametrize("sec_units", [3584 * 2 + 1561, 3584 + 217, 448 * 4 + 100, 3584 * 3])
def test_partial_last_tiles_with_divergent_warps(sec_units, dtype):
    """Geometry of the full-size configs at small scale: sections of several 3584-unit tiles plus a partial last tile
    whose last streaming round is entered by only some lanes of a warp (the others take the remainder path).  The
    dead-source discard must not drop a line whose other vectors are loaded by a later instruction: outputs and masks
    are compared with the oracle bit for bit."""
    p, k = 5, 4
    A = 4 if dtype == W.F32 else 8
    n = (p - 1) * k * sec_units * A
    w = _wl(p, 1, {0: 2.0}, n, dtype, seed=77)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=B.OPTCC_EXEC_DATAFLOW, tile_units=3584)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    x = W.all_inputs(w)
    s = _session(plan, verify=True)
    s.upload(x)
    s.execute()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    res = s.verify()
    assert res["bad_elements"] == 0 and res["overlap_elements"] == 0


def test_discard_can_be_disabled_and_changes_nothing():
    w = _wl(8, 1, {0: 2.0}, 4 * 7 * 4 * (3584 + 300), W.F32, seed=13)
    outs = []
    for nd in (0, 1):
        plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4, exec_mode=B.OPTCC_EXEC_DATAFLOW, tile_units=3584, no_discard=nd)
        s = _session(plan)
        s.upload(W.all_inputs(w))
        s.execute()
        outs.append(s.download().tobytes())
    assert outs[0] == outs[1]


def test_truncated_schedule_midsize_masks_equal_oracle():
    """A truncated schedule at a size where full streaming rounds run: the masks must still equal the oracle's for
    the same truncated table (so nothing may be dropped from L2 on the assumption that a later step overwrites it)."""
    import dataclasses
    p, k, limit = 5, 4, 9
    n = 4 * (p - 1) * k * (3584 + 300)
    ell = [1.0, 1.0, 2.0, 1.0, 1.0]
    plan = B.optcc_plan(p, 1, ell, n, W.F32, k=k, exec_mode=B.OPTCC_EXEC_DATAFLOW, step_limit=limit, tile_units=3584)
    oplan = OP.build_plan(p, 1, ell, n, W.F32, k=k)
    s = _session(plan, verify=True)
    res = s.verify(raise_on_fail=False)
    m_or, _ = OI.element_masks(dataclasses.replace(oplan, n_steps=limit))
    assert s.masks().tobytes() == m_or.tobytes()
    assert res["bad_elements"] == int((m_or != OI.full_mask_words(p)[None, None, :]).any(axis=2).sum()) > 0


def _oracle_prefix(oplan, limit):
    """the oracle's plan cut after `limit` steps: the table rows of steps < limit (PLAN_SPEC 3: step_begin)"""
    import dataclasses
    return dataclasses.replace(oplan, n_steps=limit, flows=oplan.flows[:int(oplan.step_begin[limit])],
                               step_begin=oplan.step_begin[:limit + 1])


TRUNC_CASES = [
    # p, g, stragglers, n, k, tile_units (0 = auto): sizes that reach full streaming rounds and partial last rounds
    (5, 1, {2: 2.0}, 4 * 4 * 4 * (3584 + 300), 4, 3584),
    (5, 1, {2: 1.5}, 4 * 4 * 4 * (1792 + 77) + 3, 4, 0),          # bubble filling, ragged n
    (16, 1, {0: 8.0 / 7.0}, 4 * 15 * 8 * 2000, 8, 0),             # C2 shape
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 400003, 4, 0),                 # several stragglers
    (16, 4, {r: 2.0 for r in range(4)}, 4 * 4 * 3 * 4 * 1900, 4, 0),   # g > 1: collect / NIC / distribute
    (6, 1, {}, 6 * 4 * 2500 + 1, 0, 0),                           # plain ring
]


@pytest.mark.parametrize("exec_mode", MODES)
@pytest.mark.parametrize("case", range(len(TRUNC_CASES)))
def test_truncated_schedule_data_equals_oracle_prefix(case, exec_mode):
    """"Steps exactly as the plan lists them" (north_star; PAPER.md:138 data dependencies), made observable: after the
    first t steps (opts.step_limit = t) EVERY element of EVERY rank buffer must hold exactly what the oracle holds
    after walking the table rows of steps < t -- the intermediate state of the p memories, not only the final one.
    In particular the column executor, which runs a tile's flows in table order without any global step order and keeps
    partial sums in registers between consecutive flows, must have stored every destination that no later EXECUTED flow
    overwrites, and nothing may have been elided or dropped from the caches on the assumption that a step beyond the
    cut overwrites it."""
    p, g, st, n, k, tile = TRUNC_CASES[case]
    w = _wl(p, g, st, n, W.F32, seed=4242 + case)
    oplan = OP.build_plan(p, g, list(w.ell), n, W.F32, k=k)
    x = W.all_inputs(w)
    rng = np.random.default_rng(900 + case)
    limits = sorted(set([1, oplan.n_steps - 1] + [int(t) for t in rng.integers(1, oplan.n_steps, size=3)]))
    for limit in limits:
        plan = B.optcc_plan(p, g, w.ell, n, W.F32, k=k, exec_mode=exec_mode, step_limit=limit, tile_units=tile)
        s = _session(plan)
        s.upload(x)
        s.execute()
        y = s.download()
        y_or = OI.run_f32(_oracle_prefix(oplan, limit), x)
        assert y.tobytes() == y_or.tobytes(), f"state after {limit} of {oplan.n_steps} steps differs from the oracle's"
        del s, plan


@pytest.mark.parametrize("exec_mode", [B.OPTCC_EXEC_COLUMN, B.OPTCC_EXEC_DATAFLOW])
def test_truncated_schedule_data_at_c2_full_size(exec_mode):
    """the same at BASELINE.json configs[1] (n = 2^26, bench.py's k): sampled elements of every rank against the
    oracle's walk of the table prefix, for a cut inside the pipeline (some sections reduced, some already gathered)"""
    import torch
    w = W.config(1)
    k = 16
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    limit = (oplan.n_steps * 3) // 5 + 4
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=exec_mode, step_limit=limit)
    s = _session(plan)
    x = W.all_inputs(w)
    s.upload(x)
    s.execute()
    torch.cuda.synchronize()
    idx = W.sample_indices(w, 1024)
    ti = torch.from_numpy(idx).to(s.device)
    ys = np.stack([s.bufs[r][ti].cpu().numpy() for r in range(w.p)])
    y_or = OI.run_f32_at(_oracle_prefix(oplan, limit), np.ascontiguousarray(x[:, idx]), idx)
    assert ys.tobytes() == y_or.tobytes()
    assert not np.array_equal(ys[0], ys[1])      # (the cut really is mid-schedule: the ranks still differ)


@pytest.mark.parametrize("exec_mode", MODES)
def test_a_clobbered_workspace_is_detected_not_executed(exec_mode):
    """optcc.h "Workspace contract": the library remembers which plan's tables a workspace holds.  If the caller reuses
    that memory in between, a later launch must not walk whatever it finds there: every kernel compares the stamp
    written with the tables and does nothing when it differs; optcc_workspace_check / optcc_verify report ESTALE, and
    after optcc_prepare everything works again."""
    import torch
    w = _wl(8, 1, {3: 1.5}, 300007, W.F32, seed=31)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4, exec_mode=exec_mode)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=4)
    x = W.all_inputs(w)
    s = _session(plan, verify=True)
    s.upload(x)
    s.prepare()
    torch.cuda.synchronize()
    s.workspace.random_(0, 255)             # the caller used the memory for something else
    s.execute()                             # (the library still believes the tables are there: no re-upload)
    torch.cuda.synchronize()
    assert s.download().tobytes() == x.tobytes()          # nothing was executed
    with pytest.raises(B.OptccError) as e:
        s.check()
    assert e.value.name == "ESTALE"
    with pytest.raises(B.OptccError) as e:
        s.verify()
    assert e.value.name == "ESTALE"
    s.prepare()                             # tables and stamp written again
    s.execute()
    s.check()
    assert s.download().tobytes() == OI.run_f32(oplan, x).tobytes()
    assert s.verify()["bad_elements"] == 0


@pytest.mark.parametrize("n_shards", [2, 3, 7])
@pytest.mark.parametrize("dtype", [W.F32, W.BF16])
def test_the_shards_of_the_work_items_together_are_the_whole_allreduce(n_shards, dtype):
    """optcc_execute_shard (include/optcc.h "ranks on several GPUs"): shard s of S runs the work items i = s (mod S); run
    one after another in ONE process on the same buffers, the S shards leave exactly optcc_execute's result, and the S
    optcc_verify_shard calls check every element once."""
    import torch
    w = _wl(16, 1, {0: 8.0 / 7.0}, 2 ** 19 + 6, dtype, seed=61)
    plan = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4)
    oplan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=4)
    x = W.all_inputs(w)
    s = _session(plan, verify=True)
    s.upload(x)
    stream = torch.cuda.current_stream().cuda_stream
    for shard in reversed(range(n_shards)):            # any order: the shards touch disjoint element columns
        B.optcc_execute_shard(plan, s.bufs, s.ws_ptr, shard, n_shards, stream)
    torch.cuda.synchronize()
    y = s.download()
    y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
    assert y.tobytes() == y_or.tobytes()
    checked = 0
    for shard in range(n_shards):
        v = B.optcc_verify_shard(plan, s.ws_ptr, shard, n_shards, stream)
        assert v["bad_elements"] == 0 and v["overlap_elements"] == 0
        checked += v["checked"]
    assert checked == w.p * w.n
    with pytest.raises(B.OptccError):
        B.optcc_execute_shard(plan, s.bufs, s.ws_ptr, n_shards, n_shards, stream)      # shard out of range
    plan_df = B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=4, exec_mode=B.OPTCC_EXEC_DATAFLOW)
    with pytest.raises(B.OptccError) as e:
        B.optcc_execute_shard(plan_df, s.bufs, s.ws_ptr, 0, 2, stream)                 # only the column executor shards
    assert e.value.code == B.OPTCC_EUNSUPPORTED
