"""oracle/walk.c (the compiled CPU baseline's walk) against oracle.interpreter.run_f32, bit for bit, and against what
the mathematics fixes: small integers sum exactly in any order, so every rank must end with the plain sum."""
import numpy as np
import pytest

from oracle import cwalk, interpreter as OI, planner as OP

CASES = [
    (4, 1, {0: 2.0}, 4099, 8, {}),
    (5, 1, {2: 1.5}, 50001, 4, {}),                                   # bubble filling
    (16, 1, {0: 8.0 / 7.0}, 2 ** 14 + 2, 8, {}),
    (6, 1, {}, 7777, 0, {}),                                          # plain ring
    (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 6553, 4, {}),
    (16, 4, {r: 2.0 for r in range(4)}, 40001, 4, {}),
    (9, 1, {4: 3.0}, 12345, 8, {"ordering": 3}),
    (16, 1, {3: 4.0 / 3.0}, 20001, 0, {"schedule": 1}),
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_c_walk_equals_the_numpy_walk(case):
    p, g, st, n, k, extra = CASES[case]
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    plan = OP.build_plan(p, g, ell, n, 0, k=k, **extra)
    rng = np.random.default_rng(40 + case)
    x = rng.standard_normal((p, n)).astype(np.float32)
    y = cwalk.run_f32(plan, x)
    assert y.tobytes() == OI.run_f32(plan, x).tobytes()
    xi = rng.integers(-1000, 1000, size=(p, n)).astype(np.float32)     # exact in fp32 whatever the order
    yi = cwalk.run_f32(plan, xi)
    assert (yi == xi.sum(axis=0, dtype=np.float64).astype(np.float32)[None, :]).all()


def test_c_walk_rejects_a_record_out_of_range():
    plan = OP.build_plan(4, 1, [2.0, 1.0, 1.0, 1.0], 4099, 0, k=4)
    import dataclasses
    flows = plan.flows.copy()
    flows["off"][3] = plan.n            # a range beyond the buffer
    with pytest.raises(ValueError):
        cwalk.run_f32(dataclasses.replace(plan, flows=flows), np.zeros((4, 4099), dtype=np.float32))
    assert cwalk.threads() >= 1
