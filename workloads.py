"""Seeded synthetic inputs shared by the tests, bench.py and the oracle's timing leg.

This module holds NONE of the method's arithmetic: it only draws the input
matrices of PAPER.md eq. (15) (section 3.2),

    a_ij, b_ij = (rand - 0.5) * exp(phi * randn),

and the structured matrices of the paper's worked example (all-ones times a
scalar alpha).  Both the CUDA path and the oracle receive the very
same arrays.

Recipe: numpy.random.Generator(PCG64(seed)),
float64; draw order U for A, Z for A, U for B, Z for B; every draw fills its
matrix in column-major (Fortran) order; seed = 29129000 + 10*config + variant.
"""
from __future__ import annotations

import numpy as np

SEED_BASE = 29129000

# BASELINE.json `configs`, restated.  `moduli` is the
# sweep the config names; `phi` the spread parameter of eq. (15).
CONFIGS = {
    0: dict(name="cfg0_128", m=128, n=128, k=128, phi=0.5, moduli=(14,)),
    1: dict(name="cfg1_1024", m=1024, n=1024, k=1024, phi=1.0, moduli=tuple(range(8, 21))),
    2: dict(name="cfg2_8192", m=8192, n=8192, k=8192, phi=0.5, moduli=tuple(range(14, 19))),
    3: dict(name="cfg3_16384", m=16384, n=16384, k=16384, phi=4.0, moduli=tuple(range(16, 21))),
    4: dict(name="cfg4_longk", m=4096, n=4096, k=65536, phi=1.0, moduli=tuple(range(14, 21))),
}

# Scale-invariance variant of config 1 (BASELINE.json configs[1]).
SCALE_CONSTANTS = (2.0 ** -500, 1e-100, 1.0, 1e100, 2.0 ** 500)


def seed_for(config: int, variant: int = 0) -> int:
    return SEED_BASE + 10 * int(config) + int(variant)


def eq15_matrices(m: int, n: int, k: int, phi: float, seed: int):
    """A (m x k) and B (k x n), float64, column-major, drawn per eq. (15)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    # draw order: U_A, Z_A, U_B, Z_B; element t of a stream is entry (t % rows, t // rows)
    ua = rng.random(m * k)
    za = rng.standard_normal(m * k)
    ub = rng.random(k * n)
    zb = rng.standard_normal(k * n)
    a = ((ua - 0.5) * np.exp(phi * za)).reshape((k, m)).T
    b = ((ub - 0.5) * np.exp(phi * zb)).reshape((n, k)).T
    return np.asfortranarray(a), np.asfortranarray(b)


def config_matrices(config: int, variant: int = 0, *, shape=None):
    """Matrices of BASELINE config `config`; `shape=(m, n, k)` overrides the size
    (used for row/column slabs that keep the config's distribution)."""
    c = CONFIGS[config]
    m, n, k = shape if shape is not None else (c["m"], c["n"], c["k"])
    return eq15_matrices(m, n, k, c["phi"], seed_for(config, variant))


def all_ones_scaled(m: int, n: int, k: int, alpha: float):
    """A = alpha * ones(m, k), B = alpha * ones(k, n)  (paper's worked example)."""
    a = np.full((m, k), float(alpha), dtype=np.float64, order="F")
    b = np.full((k, n), float(alpha), dtype=np.float64, order="F")
    return a, b


def small_integer_matrices(m: int, n: int, k: int, bound: int, seed: int):
    """Integer-valued float64 matrices with |entry| <= bound (textbook special case:
    the emulated product must equal the exact integer matmul)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    a = rng.integers(-bound, bound + 1, size=(k, m)).T.astype(np.float64)
    b = rng.integers(-bound, bound + 1, size=(n, k)).T.astype(np.float64)
    return np.asfortranarray(a), np.asfortranarray(b)


def wide_exponent_matrices(m: int, n: int, k: int, seed: int, zero_fraction: float = 0.05):
    """Stress inputs for the integer stages: random signs and mantissas with exponents
    spread over the whole normal and subnormal FP64 range inside each matrix, some exact
    zeros, one all-zero row of A and one all-zero column of B."""
    rng = np.random.Generator(np.random.PCG64(seed))

    def one(rows, cols):
        mant = rng.random(rows * cols) + 1.0
        ex = rng.integers(-1070, 500, size=rows * cols)
        sgn = rng.integers(0, 2, size=rows * cols) * 2.0 - 1.0
        v = sgn * np.ldexp(mant, ex)
        v[rng.random(rows * cols) < zero_fraction] = 0.0
        return v

    a = one(m, k).reshape((k, m)).T.copy()
    b = one(k, n).reshape((n, k)).T.copy()
    if m > 1:
        a[m // 2, :] = 0.0
    if n > 1:
        b[:, n // 3] = 0.0
    return np.asfortranarray(a), np.asfortranarray(b)
