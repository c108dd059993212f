"""Pins for the arithmetic walks of oracle/interpreter.py and the predicates of oracle/reference.py."""
import numpy as np
import pytest
import torch

from oracle import interpreter, reference
from oracle import planner as P
from paper_2606_01680_b200 import workloads as W


def ell_vec(p, d):
    return [float(d.get(i, 1.0)) for i in range(p)]


CASES = [
    (4, 1, {0: 2.0}, 1003),
    (5, 1, {3: 1.5}, 2050),
    (6, 1, {}, 777),
    (7, 1, {0: 2.0, 4: 4.0 / 3.0}, 1500),
    (8, 2, {2: 2.0, 3: 2.0}, 1234),
    (12, 4, {8: 1.5, 9: 1.5, 10: 1.5, 11: 1.5}, 999),
]


@pytest.mark.parametrize("p,g,ells,n", CASES)
def test_f32_walk_is_exact_on_integers_and_all_ranks_identical(p, g, ells, n):
    # with small integer inputs every fp32 add is exact, so any association order gives the exact sum (:68 (ii))
    plan = P.build_plan(p, g, ell_vec(p, ells), n, P.F32, k=4)
    rng = np.random.default_rng(7)
    x = rng.integers(-1000, 1000, size=(p, n)).astype(np.float32)
    y = interpreter.run_f32(plan, x)
    want = x.astype(np.int64).sum(axis=0)
    assert (y.astype(np.int64) == want[None, :]).all()
    assert reference.all_ranks_identical(y)


@pytest.mark.parametrize("p,g,ells,n", CASES)
def test_f32_walk_within_north_star_bound(p, g, ells, n):
    plan = P.build_plan(p, g, ell_vec(p, ells), n, P.F32, k=4)
    rng = np.random.default_rng(11)
    x = rng.standard_normal((p, n)).astype(np.float32)
    y = interpreter.run_f32(plan, x)
    assert reference.all_ranks_identical(y)
    assert reference.check_f32(y[0], x).all()
    # the bound is not vacuous: a dropped contributor fails it
    y_bad = y[0] - x[1]
    assert not reference.check_f32(y_bad, x).all()


def test_reference_sum_is_the_plain_definition():
    x = np.array([[1e8, 1.0], [-1e8, 2.0], [1.0, 3.0]], dtype=np.float32)
    assert reference.reference_sum(x).tolist() == [1.0, 6.0]           # fp64 keeps what fp32 would lose
    assert reference.abs_sum(x).tolist() == [2e8 + 1.0, 6.0]
    assert reference.f32_bound(x)[1] == 3 * 2.0 ** -23 * 6.0


def test_bf16_conversions_against_torch():
    # independent library routine: torch's CPU bf16 cast (RNE)
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.standard_normal(20000).astype(np.float32) * 10.0 ** rng.integers(-6, 6, 20000),
                        np.array([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 65504.0, 3.0e38, 1e-40, -1e-40], np.float32)]).astype(np.float32)
    bits = interpreter.f32_to_bf16_bits(x)
    tb = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert (bits == tb).all()
    back = interpreter.bf16_bits_to_f32(bits)
    tback = torch.from_numpy(tb.view(np.int16)).view(torch.bfloat16).to(torch.float32).numpy()
    assert (back.view(np.uint32) == tback.view(np.uint32)).all()
    # ties to even, by hand: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> 1; 1 + 3*2^-8 -> 1 + 2^-6
    assert interpreter.bf16_bits_to_f32(interpreter.f32_to_bf16_bits(np.float32(1.00390625))) == 1.0
    assert interpreter.bf16_bits_to_f32(interpreter.f32_to_bf16_bits(np.float32(1.01171875))) == 1.015625
    # the workload generator's input conversion agrees (it is a storage conversion, not method arithmetic)
    assert (W._rne_bf16_bits(x[:20000].copy()) == bits[:20000]).all()


@pytest.mark.parametrize("p,g,ells,n", CASES)
def test_bf16_walk_single_final_rounding(p, g, ells, n):
    plan = P.build_plan(p, g, ell_vec(p, ells), n, P.BF16, k=4)
    rng = np.random.default_rng(5)
    xb = interpreter.f32_to_bf16_bits(rng.standard_normal((p, n)).astype(np.float32))
    x32 = interpreter.bf16_bits_to_f32(xb)
    yb = interpreter.run_bf16(plan, xb)
    assert reference.all_ranks_identical(yb)
    y32 = interpreter.bf16_bits_to_f32(yb[0])
    assert reference.check_bf16(y32, x32).all()                       # R12
    # equals: fp32 sum in the same plan order, then ONE rounding
    plan32 = P.build_plan(p, g, ell_vec(p, ells), n, P.BF16, k=4)
    y_f32_order = interpreter.run_f32(plan32, x32)
    assert (interpreter.f32_to_bf16_bits(y_f32_order[0]) == yb[0]).all()
    # small integers: exact
    xi = rng.integers(-3, 4, size=(p, n)).astype(np.float32)
    yi = interpreter.run_bf16(plan, interpreter.f32_to_bf16_bits(xi))
    assert (interpreter.bf16_bits_to_f32(yi[0]) == xi.sum(axis=0)).all()


def test_per_hop_bf16_rounding_would_fail_the_bound():
    # SURVEY §7 "Hard parts": rounding the partial at every hop breaks 2^-7; one final rounding does not.
    p, n = 64, 4096
    rng = np.random.default_rng(2)
    xb = interpreter.f32_to_bf16_bits(rng.standard_normal((p, n)).astype(np.float32))
    x32 = interpreter.bf16_bits_to_f32(xb)
    acc = x32[0].copy()
    for i in range(1, p):
        acc = interpreter.bf16_bits_to_f32(interpreter.f32_to_bf16_bits(acc + x32[i]))
    assert reference.count_bf16_pure_relative_failures(acc, x32) > n // 10
    one = interpreter.bf16_bits_to_f32(interpreter.f32_to_bf16_bits(x32.sum(axis=0, dtype=np.float32)))
    assert reference.check_bf16(one, x32).all()


def test_workload_generators_are_seeded_and_sliceable():
    w = W.config(0).scaled(5000)
    a = W.rank_input(w, 2)
    b = W.rank_input(w, 2)
    assert (a == b).all() and a.dtype == np.float32 and -1.0 <= a.min() and a.max() < 1.0
    assert (W.rank_input(w, 2, 100, 200) == a[100:200]).all()
    assert not (W.rank_input(w, 3) == a).all()
    w3 = W.config(2).scaled(4096)
    xb = W.rank_input(w3, 5)
    assert xb.dtype == np.uint16 and abs(float(interpreter.bf16_bits_to_f32(xb).std()) - 1.0) < 0.1
    w2 = W.config(1).scaled(20000)
    assert abs(float(W.rank_input(w2, 0).std()) - 0.1) < 0.01           # R15: variance 1e-2
    for i in range(5):
        c = W.config(i)
        assert len(c.ell) == c.p
    idx = W.sample_indices(W.config(1), 100)
    assert idx[0] == 0 and idx[-1] == 2 ** 26 - 1 and len(idx) <= 100
