"""Pins for the oracle's SGEMM variant (FP32 in / FP32 out; Fig. 6): the final rounding is
RN_32 of the exact integer (one rounding), Steps 1-3 are the FP64 path on the promoted inputs."""
import math
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O

ACCU, FAST, PROP = 0, 1, 2


def rn32(x: Fraction) -> np.float32:
    """correctly rounded float32 of an exact rational (ties to even), via exact comparison of the two neighbours"""
    if x == 0:
        return np.float32(0.0)
    if abs(x) >= Fraction(2) ** 128 - Fraction(2) ** 103:       # rounds to +-inf
        return np.float32(np.inf if x > 0 else -np.inf)
    if abs(x) >= Fraction(2) ** 127:                             # top binade: float(x) -> float32 cast is safe, neighbours may be inf
        lo = Fraction(2) ** 104
        q = x / lo
        n = q.numerator // q.denominator
        rem = q - n
        n += 1 if (rem > Fraction(1, 2) or (rem == Fraction(1, 2) and n % 2)) else 0
        return np.float32(float(n * lo))
    f = np.float32(float(x))                      # float(x) is RN_64; may double-round: fix with exact neighbours
    cands = [np.nextafter(f, np.float32(-np.inf)), f, np.nextafter(f, np.float32(np.inf))]
    best = min(cands, key=lambda c: (abs(Fraction(float(c)) - x), int(np.float32(c).view(np.uint32)) & 1))
    return np.float32(best)


def test_words_to_float_is_correctly_rounded_single_rounding():
    rng = np.random.Generator(np.random.PCG64(5))
    for _ in range(400):
        bits = int(rng.integers(1, 150))
        v = int(rng.integers(0, 2 ** 62)) << max(0, bits - 62) | int(rng.integers(0, 2))
        v = v if rng.random() < 0.5 else -v
        sh = int(rng.integers(-200, 60))
        assert O.words_to_float(O.int_to_words(v), sh) == rn32(Fraction(v) * Fraction(2) ** sh), (v, sh)
    # double-rounding trap: 2^24 + 1 + 2^-30 must round UP to 2^24 + 2 (RN_64 first would give the tie 2^24 + 1 -> even)
    v = (2 ** 24 + 1) * 2 ** 60 + 2 ** 30
    assert O.words_to_float(O.int_to_words(v), -60) == np.float32(2 ** 24 + 2)
    # subnormal FP32 results round once, overflow gives inf
    assert O.words_to_float(O.int_to_words(3), -150) == rn32(Fraction(3, 2 ** 150))
    assert np.isinf(O.words_to_float(O.int_to_words(1), 128))


@pytest.mark.parametrize("mode", [ACCU, FAST, PROP])
def test_small_integer_matrices_exact(mode):
    A, B = W.small_integer_matrices(24, 20, 40, 8, 3)
    C = O.sgemm(A, B, 8, mode)
    assert C.dtype == np.float32 and np.array_equal(C.astype(np.float64), A @ B)


@pytest.mark.parametrize("mode", [ACCU, PROP])
def test_final_value_is_rn32_of_the_exact_scaled_integer_product(mode):
    A, B = W.eq15_matrices(12, 10, 64, 1.0, 9)
    A, B = A.astype(np.float32), B.astype(np.float32)
    N = 10
    C, e, f = O.sgemm(A, B, N, mode, return_exponents=True)
    # exact A'B' in Python integers with the oracle's exponents, one rounding to FP32
    def tr(v, ex):
        return math.trunc(Fraction(float(v)) * Fraction(2) ** int(ex))

    for i in range(12):
        for j in range(10):
            z = sum(tr(A[i, h], e[i]) * tr(B[h, j], f[j]) for h in range(64))
            assert C[i, j] == rn32(Fraction(z) / Fraction(2) ** (int(e[i]) + int(f[j]))), (i, j)


def test_same_exponents_as_the_fp64_path_on_promoted_inputs_and_alpha_beta():
    A, B = W.eq15_matrices(20, 16, 100, 0.5, 4)
    A, B = A.astype(np.float32), B.astype(np.float32)
    C, e, f = O.sgemm(A, B, 9, PROP, return_exponents=True)
    e2, f2 = O.exponents(PROP, 9, A.astype(np.float64), B.astype(np.float64))
    assert np.array_equal(e, e2) and np.array_equal(f, f2)
    rng = np.random.Generator(np.random.PCG64(2))
    Cin = rng.standard_normal((20, 16)).astype(np.float32)
    out = O.sgemm(A, B, 9, PROP, alpha=0.75, beta=-1.5, C_in=Cin)
    t = (np.float32(0.75) * C).astype(np.float32)
    want = (np.float64(-1.5) * Cin.astype(np.float64) + t.astype(np.float64)).astype(np.float32)   # fmaf: exact then one rounding
    assert np.array_equal(out, want)


def test_accuracy_reaches_fp32_level_with_few_moduli():
    # SGEMM needs N = 3..12 moduli; with enough moduli the error is the FP32 rounding of the result
    A, B = W.eq15_matrices(32, 32, 256, 0.5, 8)
    A, B = A.astype(np.float32), B.astype(np.float32)
    ref = A.astype(np.float64) @ B.astype(np.float64)
    errs = {N: np.max(np.abs(O.sgemm(A, B, N, PROP).astype(np.float64) - ref) / np.abs(ref)) for N in (4, 6, 8, 10)}
    assert errs[4] > 10 * errs[6] > 10 * errs[8]
    assert errs[10] <= 2.0 ** -24


def test_unscale_f32_is_rn32_of_the_scaled_integer_then_fp32_alpha_beta():
    # the FP32 tail on its own (used by the GPU CRT boundary tests): RN_32(z 2^-(e+f)) from exact rationals,
    # then t = RN_32(alpha c), out = RN_32(beta C_in + t) (fmaf)
    rng = np.random.Generator(np.random.PCG64(17))
    n, m = 3, 7
    zs = [[int(rng.integers(-2 ** 62, 2 ** 62)) * (1 << int(rng.integers(0, 60))) + int(rng.integers(-5, 5)) for _ in range(m)]
          for _ in range(n)]
    Cpp = np.stack([np.stack([O.int_to_words(z) for z in row]) for row in zs])
    e = rng.integers(20, 90, size=m).astype(np.int32)
    f = rng.integers(20, 90, size=n).astype(np.int32)
    got = O.unscale_f32(Cpp, e, f)
    assert np.all(np.isfinite(got))
    for j in range(n):
        for i in range(m):
            assert got[i, j] == rn32(Fraction(zs[j][i]) / Fraction(2) ** (int(e[i]) + int(f[j]))), (i, j)
    Cin = rng.standard_normal((m, n)).astype(np.float32)
    out = O.unscale_f32(Cpp, e, f, alpha=0.75, beta=-1.5, C_in=Cin)
    for j in range(n):
        for i in range(m):
            t = rn32(Fraction(0.75) * Fraction(float(got[i, j])))
            assert out[i, j] == rn32(Fraction(-1.5) * Fraction(float(Cin[i, j])) + Fraction(float(t))), (i, j)
