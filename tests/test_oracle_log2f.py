"""Pins for LOG2F, the oracle's stand-in for __log2f on [1,2] (reading R3).

The definition is mathematical: LOG2F(x) = RN_32(log2 x).  It is pinned against 200-bit
mpmath (random inputs, the inputs closest to a rounding midpoint, the interval ends), the
paper's error model |__log2f(x) - log2 x| <= 4 u32 on [0.5, 2], and
exhaustively over all 2^23 + 1 floats of [1, 2] against a different libm routine.
"""
import numpy as np
from mpmath import mp, mpf, log

from oracle import ozaki2_oracle as O

U32 = 2.0 ** -24


def _rn32(x):
    """mpf -> nearest float32 (ties to even; ties do not occur for log2 of a float != 1, 2)."""
    f = np.float32(float(x))          # double rounding is harmless: checked by the margin below
    lo = np.nextafter(f, np.float32(-np.inf))
    hi = np.nextafter(f, np.float32(np.inf))
    best = min((lo, f, hi), key=lambda c: abs(mpf(float(c)) - x))
    return np.float32(best)


def _all_floats_in_1_2():
    bits = np.arange(0x3F800000, 0x40000000 + 1, dtype=np.uint32)
    return bits.view(np.float32)


def test_log2f_exhaustive_vs_second_libm_and_error_model():
    x = _all_floats_in_1_2()
    y = O.log2f_array(x)
    # a different routine: numpy's FP64 log2, rounded once to FP32
    y2 = np.log2(x.astype(np.float64)).astype(np.float32)
    assert np.array_equal(y, y2)
    # paper's error model, P:145 / P:330: absolute error <= 4 u32 on [0.5, 2]
    err = np.abs(y.astype(np.float64) - np.log2(x.astype(np.float64)))
    assert err.max() <= 4 * U32
    assert err.max() <= U32                    # in fact at most half an ulp of a value in [0,1]
    assert y[0] == 0.0 and y[-1] == 1.0        # LOG2F(1) = 0, LOG2F(2) = 1 exactly
    assert np.all(np.diff(y) >= 0)             # monotone


def test_log2f_correctly_rounded_mpmath():
    mp.prec = 200
    rng = np.random.Generator(np.random.PCG64(5))
    x = _all_floats_in_1_2()
    # the hardest inputs: FP64 log2 closest to a float32 rounding midpoint
    y64 = np.log2(x.astype(np.float64))
    y32 = y64.astype(np.float32)
    up = np.nextafter(y32, np.float32(2))
    dn = np.nextafter(y32, np.float32(-1))
    mid_hi = (y32.astype(np.float64) + up.astype(np.float64)) / 2
    mid_lo = (y32.astype(np.float64) + dn.astype(np.float64)) / 2
    ulp = (up.astype(np.float64) - y32.astype(np.float64))
    dist = np.minimum(np.abs(y64 - mid_hi), np.abs(y64 - mid_lo)) / np.maximum(ulp, 1e-300)
    hard = np.argsort(dist)[:300]
    sample = np.concatenate([hard, rng.integers(0, x.size, 3000), [0, 1, 2, x.size - 2, x.size - 1]])
    for t in sample:
        xv = x[int(t)]
        want = _rn32(log(mpf(float(xv)), 2))
        assert O.log2f(xv) == want, float(xv)
