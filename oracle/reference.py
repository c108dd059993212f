"""Result definition and tolerance predicates (PAPER.md:68 (ii); BASELINE.json north_star).

Test infrastructure only (see oracle/__init__.py).
"""
import numpy as np


def reference_sum(x):
    """y_ref[e] = sum_i (double) x_i[e]  (:68 (ii)), x[p, n] float32 (or fp32 values of bf16 data)."""
    return np.sum(np.asarray(x, dtype=np.float64), axis=0, dtype=np.float64)


def abs_sum(x):
    """sum_i |x_i[e]| in fp64 (the scale of the fp32 bound)."""
    return np.sum(np.abs(np.asarray(x, dtype=np.float64)), axis=0, dtype=np.float64)


def f32_bound(x):
    """north_star: |y - y_ref| <= p 2^-23 sum_i |x_i| per element."""
    p = np.asarray(x).shape[0]
    return p * 2.0 ** -23 * abs_sum(x)


def check_f32(y, x):
    """Boolean array: which elements of fp32 output y meet the fp32 bound."""
    err = np.abs(np.asarray(y, dtype=np.float64) - reference_sum(x))
    return err <= f32_bound(x)


def check_bf16(y_f32, x_f32):
    """R12: |y - y_ref| <= 2^-7 |y_ref| + p 2^-23 sum|x_i|  (relative term + fp32 accumulation floor).
    y_f32: the bf16 outputs widened to fp32; x_f32: the bf16 inputs widened to fp32, [p, n]."""
    ref = reference_sum(x_f32)
    err = np.abs(np.asarray(y_f32, dtype=np.float64) - ref)
    return err <= 2.0 ** -7 * np.abs(ref) + f32_bound(x_f32)


def count_bf16_pure_relative_failures(y_f32, x_f32):
    """Number of elements failing the pure 2^-7 relative test (reported, not gating; R12)."""
    ref = reference_sum(x_f32)
    err = np.abs(np.asarray(y_f32, dtype=np.float64) - ref)
    return int(np.count_nonzero(err > 2.0 ** -7 * np.abs(ref)))


def all_ranks_identical(y):
    """:68 (ii): every GPU holds the same vector -- bitwise (compare raw bytes, so NaN == NaN and -0 != 0)."""
    y = np.ascontiguousarray(y)
    raw = y.view(np.uint8).reshape(y.shape[0], -1)
    return bool((raw == raw[0]).all())
