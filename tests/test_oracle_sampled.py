"""The sampled walks run_f32_at / run_bf16_at (used by the full-size GPU parity tests) equal the full walks
run_f32 / run_bf16 -- which are pinned in test_oracle_numerics.py -- restricted to the sample."""
import numpy as np
import pytest

from oracle import planner as OP
from oracle import interpreter as OI

CASES = [
    (4, 1, {0: 2.0}, 4099, 8), (5, 1, {2: 1.5}, 50001, 4), (6, 1, {}, 7777, 0), (7, 1, {0: 2.0, 1: 4.0 / 3.0}, 20011, 4),
    (16, 4, {r: 2.0 for r in range(4)}, 40001, 4), (64, 1, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}, 9001, 4),
]


@pytest.mark.parametrize("p,g,st,n,k", CASES)
@pytest.mark.parametrize("dtype", [OP.F32, OP.BF16])
def test_sampled_walk_equals_full_walk(p, g, st, n, k, dtype):
    ell = [float(st.get(i, 1.0)) for i in range(p)]
    plan = OP.build_plan(p, g, ell, n, dtype, k=k)
    rng = np.random.default_rng(p * 1000 + n)
    idx = np.unique(np.concatenate([rng.integers(0, n, size=257), [0, n - 1]]))
    x = rng.standard_normal((p, n)).astype(np.float32)
    if dtype == OP.F32:
        full = OI.run_f32(plan, x)
        part = OI.run_f32_at(plan, x[:, idx], idx)
        assert part.tobytes() == np.ascontiguousarray(full[:, idx]).tobytes()
    else:
        xb = OI.f32_to_bf16_bits(x)
        full = OI.run_bf16(plan, xb)
        part = OI.run_bf16_at(plan, xb[:, idx], idx)
        assert part.tobytes() == np.ascontiguousarray(full[:, idx]).tobytes()
