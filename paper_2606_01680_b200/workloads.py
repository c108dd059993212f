"""Seeded synthetic workloads: BASELINE.json's five configs and their input generators.

This module holds NO arithmetic of the method (no planning, reducing, rounding of sums); it only
describes workloads and draws inputs.  It serves both the CUDA path's tests/bench and the oracle's
tests, so that both see byte-identical inputs.  It imports neither oracle/ nor the CUDA binding.

Inputs stand in for the paper's data-parallel gradient buffers ("hundreds of MB to several GB",
PAPER.md:58; p in [16,256], l in {8/7, 4/3, 2}, g in {4, 8}); the paper uses no
public dataset.  Generator: numpy Generator(PCG64(SeedSequence([seed, rank]))), one stream per rank.
"""
from dataclasses import dataclass, field
from typing import List

import numpy as np

F32, BF16 = 0, 1


@dataclass(frozen=True)
class Workload:
    name: str
    p: int
    g: int
    ell: tuple          # length p
    n: int
    dtype: int          # F32 | BF16
    dist: str           # "uniform" U[-1,1) | "normal"
    sigma: float        # std-dev for "normal"
    seed: int
    note: str = ""

    @property
    def elem_bytes(self):
        return 4 if self.dtype == F32 else 2

    def scaled(self, n, name=None):
        """Same workload shape with a different per-rank length (parity-test sizes)."""
        return Workload(name or f"{self.name}@n={n}", self.p, self.g, self.ell, n, self.dtype,
                        self.dist, self.sigma, self.seed, self.note)


def _ell(p, d):
    return tuple(float(d.get(i, 1.0)) for i in range(p))


def config(i, ell_c5=1.6):
    """BASELINE.json configs[i] (i = 0..4 <-> C1..C5 of SURVEY.md §8(d))."""
    if i == 0:   # C1
        return Workload("C1", 4, 1, _ell(4, {0: 2.0}), 2 ** 20, F32, "uniform", 1.0, 0,
                        "p=4, straggler rank 0 ell=2, n=2^20 f32, U[-1,1)")
    if i == 1:   # C2
        return Workload("C2", 16, 1, _ell(16, {0: 8.0 / 7.0}), 2 ** 26, F32, "normal", 0.1, 1,
                        "p=16, straggler rank 0 ell=8/7, n=2^26 f32, N(0, var 1e-2) (R15: sigma=0.1)")
    if i == 2:   # C3
        return Workload("C3", 64, 1, _ell(64, {5: 8.0 / 7.0, 17: 4.0 / 3.0, 40: 2.0}), 2 ** 24, BF16,
                        "normal", 1.0, 2, "p=64, m=3 stragglers, n=2^24 bf16, N(0,1) drawn f32 then RNE to bf16")
    if i == 3:   # C4
        return Workload("C4", 128, 8, _ell(128, {r: 2.0 for r in range(8)}), 2 ** 22, F32, "uniform", 1.0, 3,
                        "g=8 x 16 servers, server 0 ell=2, n=2^22 f32, U[-1,1)")
    if i == 4:   # C5 (one ell of the sweep)
        return Workload(f"C5[ell={ell_c5:.6g}]", 32, 1, _ell(32, {0: float(ell_c5)}), 2 ** 25, F32,
                        "normal", 1.0, 4, "p=32, straggler rank 0, ell swept, n=2^25 f32, N(0,1)")
    raise IndexError(i)


C5_ELLS = (1.0, 8.0 / 7.0, 4.0 / 3.0, 1.6, 2.0 - 1.0 / 31.0, 2.0, 3.0)


def _rne_bf16_bits(x32):
    """Storage-format conversion of the *inputs* only: float32 -> bf16 bit pattern (RNE)."""
    u = x32.view(np.uint32)
    return ((u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)).astype(np.uint16)


def rank_input(w: Workload, rank: int, lo: int = 0, hi: int = None, out=None):
    """Elements [lo, hi) of rank `rank`'s input: float32 array (F32) or uint16 bf16 bit patterns (BF16).

    The stream is always drawn from element 0 so that any slice equals the slice of the full draw."""
    hi = w.n if hi is None else hi
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed, rank])))
    if w.dist == "uniform":
        x = rng.random(hi, dtype=np.float32)
        x *= np.float32(2.0)
        x -= np.float32(1.0)
    elif w.dist == "normal":
        x = rng.standard_normal(hi, dtype=np.float32)
        if w.sigma != 1.0:
            x *= np.float32(w.sigma)
    else:
        raise ValueError(w.dist)
    x = x[lo:hi]
    if w.dtype == BF16:
        x = _rne_bf16_bits(np.ascontiguousarray(x))
    if out is not None:
        out[...] = x
        return out
    return x


def all_inputs(w: Workload, out=None):
    """[p, n] array of all ranks' inputs (float32, or uint16 bf16 bits)."""
    dt = np.float32 if w.dtype == F32 else np.uint16
    if out is None:
        out = np.empty((w.p, w.n), dtype=dt)
    for r in range(w.p):
        rank_input(w, r, out=out[r])
    return out


def sample_indices(w: Workload, count: int, seed: int = 12345):
    """Deterministic sample of element indices in [0, n) incl. both ends (full-size sampled parity)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, w.seed, w.n])))
    idx = rng.integers(0, w.n, size=max(count - 2, 0), dtype=np.int64)
    return np.unique(np.concatenate([idx, np.array([0, w.n - 1], dtype=np.int64)]))
