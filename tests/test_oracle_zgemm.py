"""Pins for the oracle's complex variant (the paper names ZGEMM as future work without formulas, P:58, P:444;
reading in DESIGN.md 8b #4: the product of the real embeddings).  What fixes it: the textbook identity between a complex
product and its real embedding, exact integer cases, the real special case, and the paper's invariants carried over."""
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O

ACCU, FAST, PROP = 0, 1, 2


def complex_inputs(m, n, k, phi, seed):
    Ar, Br = W.eq15_matrices(m, n, k, phi, seed)
    Ai, Bi = W.eq15_matrices(m, n, k, phi, seed + 1)
    return Ar + 1j * Ai, Br + 1j * Bi


def test_embedding_is_the_complex_product_exactly_on_gaussian_integers():
    rng = np.random.Generator(np.random.PCG64(3))
    A = rng.integers(-9, 10, (7, 11)) + 1j * rng.integers(-9, 10, (7, 11))
    B = rng.integers(-9, 10, (11, 5)) + 1j * rng.integers(-9, 10, (11, 5))
    At, Bt = O.zgemm_embedding(A, B)
    Ct = At @ Bt
    want = A @ B                                           # small integers: exact in FP64
    assert np.array_equal(Ct[:7], want.real) and np.array_equal(Ct[7:], want.imag)
    # rows i and m + i of the embedded A carry the complex row's 2-norm and max-norm: one exponent per complex row
    assert np.array_equal(np.sum(At[:7] ** 2, axis=1), np.sum(At[7:] ** 2, axis=1))
    assert np.array_equal(np.sum(At[:7] ** 2, axis=1), np.sum(np.abs(A) ** 2, axis=1))


@pytest.mark.parametrize("mode", [ACCU, FAST, PROP])
def test_gaussian_integer_matrices_exact(mode):
    rng = np.random.Generator(np.random.PCG64(5))
    A = rng.integers(-8, 9, (12, 30)) + 1j * rng.integers(-8, 9, (12, 30))
    B = rng.integers(-8, 9, (30, 9)) + 1j * rng.integers(-8, 9, (30, 9))
    assert np.array_equal(O.zgemm(A, B, 10, mode), A @ B)


@pytest.mark.parametrize("mode", [FAST, PROP])
def test_real_inputs_reduce_to_dgemm_bit_for_bit(mode):
    # imaginary parts zero: the embedded rows (a, 0) and (0, a) have the statistics of the real row (zeros add nothing to
    # the max or to the rounded-up sum of squares), so the real part is oz2o_dgemm's result and the imaginary part is 0
    A, B = W.eq15_matrices(20, 14, 60, 1.0, 8)
    C = O.zgemm(A.astype(np.complex128), B.astype(np.complex128), 14, mode)
    assert np.array_equal(C.real, O.dgemm(A, B, 14, mode)) and not np.any(C.imag)


def test_both_rows_of_a_complex_row_get_the_same_exponent_and_condition_1_holds():
    A, B = complex_inputs(16, 12, 64, 1.0, 20)
    At, Bt = O.zgemm_embedding(A, B)
    for mode in (ACCU, PROP):
        e, f = O.exponents(mode, 15, At, Bt)
        if mode == PROP:
            assert np.array_equal(e[:16], e[16:])           # one scaling per complex row (P:303-311 on complex moduli)
        Ap, Bp = O.truncate(0, At, e), O.truncate(1, Bt, f)
        _, _, cnt = O.exact_product(15, Ap, Bp, want_words=False)
        assert cnt["violations"] == 0                       # P:358 / P:161-163 carried over to the embedding


def test_error_against_numpy_complex_product_and_alpha_beta():
    A, B = complex_inputs(24, 18, 128, 0.5, 30)
    ref = A @ B
    C = O.zgemm(A, B, 18, PROP)
    assert np.max(np.abs(C - ref) / np.abs(ref)) < 1e-12
    # power-of-two scale invariance of the revised mode, complex scalars of modulus 2^s included
    C2 = O.zgemm(A * 2.0 ** 40, B * (2.0 ** -70 * 1j), 18, PROP)
    assert np.array_equal(C2, C * (2.0 ** -30 * 1j))
    alpha, beta = 0.5 - 2.0j, -1.25 + 0.75j
    rng = np.random.Generator(np.random.PCG64(2))
    Cin = rng.standard_normal((24, 18)) + 1j * rng.standard_normal((24, 18))
    out = O.zgemm(A, B, 18, PROP, alpha=alpha, beta=beta, C_in=Cin)
    want = alpha * C + beta * Cin
    assert np.max(np.abs(out - want)) <= 4 * np.finfo(float).eps * np.max(np.abs(want))


def test_beta_one_adds_c_as_it_is():
    # beta == 1 is not multiplied (the BLAS rule the real entry points follow: fma(1, C, t) = C + t).  For finite C_in that
    # is the single rounding of t + C_in per part; a non-finite part of an entry stays in its own part
    A, B = complex_inputs(12, 9, 64, 0.5, 31)
    rng = np.random.Generator(np.random.PCG64(3))
    Cin = rng.standard_normal((12, 9)) + 1j * rng.standard_normal((12, 9))
    for alpha in (1.0, 0.5 - 2.0j):
        t = O.zgemm(A, B, 16, PROP, alpha=alpha)
        out = O.zgemm(A, B, 16, PROP, alpha=alpha, beta=1.0, C_in=Cin)
        for i in range(12):
            for j in range(9):                   # RN(t + c) from the exact rational sum, part by part
                for got, a, b in ((out[i, j].real, t[i, j].real, Cin[i, j].real), (out[i, j].imag, t[i, j].imag, Cin[i, j].imag)):
                    assert got == float(Fraction(float(a)) + Fraction(float(b)))
    bad = Cin.copy()
    bad[3, 4] = complex(np.inf, 2.0)
    bad[5, 6] = complex(-1.0, np.nan)
    out = O.zgemm(A, B, 16, PROP, beta=1.0, C_in=bad)
    t = O.zgemm(A, B, 16, PROP)
    assert out[3, 4].real == np.inf and out[3, 4].imag == t[3, 4].imag + 2.0
    assert out[5, 6].real == t[5, 6].real - 1.0 and np.isnan(out[5, 6].imag)
    A32, B32 = A.astype(np.complex64), B.astype(np.complex64)
    out32 = O.cgemm(A32, B32, 9, PROP, beta=1.0, C_in=bad.astype(np.complex64))
    t32 = O.cgemm(A32, B32, 9, PROP)
    assert out32.dtype == np.complex64 and out32[3, 4].real == np.inf
    assert out32[3, 4].imag == np.float32(t32[3, 4].imag + np.float32(2.0)) and np.isnan(out32[5, 6].imag)


# ---- single-precision complex variant (cgemm): the same reading on FP32 parts -------------------------------------------
def complex64_inputs(m, n, k, phi, seed):
    A, B = complex_inputs(m, n, k, phi, seed)
    return A.astype(np.complex64), B.astype(np.complex64)


@pytest.mark.parametrize("mode", [ACCU, FAST, PROP])
def test_cgemm_gaussian_integer_matrices_exact(mode):
    rng = np.random.Generator(np.random.PCG64(15))
    A = (rng.integers(-8, 9, (10, 20)) + 1j * rng.integers(-8, 9, (10, 20))).astype(np.complex64)
    B = (rng.integers(-8, 9, (20, 7)) + 1j * rng.integers(-8, 9, (20, 7))).astype(np.complex64)
    want = A.astype(np.complex128) @ B.astype(np.complex128)          # |entries| < 2^24: exact in FP32 as well
    assert np.array_equal(O.cgemm(A, B, 8, mode).astype(np.complex128), want)


@pytest.mark.parametrize("mode", [FAST, PROP])
def test_cgemm_real_inputs_reduce_to_sgemm_bit_for_bit(mode):
    A, B = W.eq15_matrices(18, 12, 50, 1.0, 9)
    A, B = A.astype(np.float32), B.astype(np.float32)
    C = O.cgemm(A.astype(np.complex64), B.astype(np.complex64), 9, mode)
    assert np.array_equal(C.real, O.sgemm(A, B, 9, mode)) and not np.any(C.imag)


def test_cgemm_is_the_single_rounding_of_zgemm_on_the_same_inputs():
    # both run Steps 1-3 on the same (exactly promoted) embedding, so C'' is the same integer: cgemm's parts are RN_32 of it,
    # zgemm's are RN_64 of it.  With enough moduli that the integer carries more than 53 significant bits nothing can be said
    # in general (double rounding), but RN_32(x) and RN_32(RN_64(x)) differ only on a 2^-29 sliver: compare within 1 ulp32
    # everywhere and bit for bit on all but a handful of entries
    A, B = complex64_inputs(20, 16, 96, 0.5, 40)
    c32 = O.cgemm(A, B, 10, PROP)
    c64 = O.zgemm(A.astype(np.complex128), B.astype(np.complex128), 10, PROP)
    for got, ref in ((c32.real, c64.real), (c32.imag, c64.imag)):
        r32 = ref.astype(np.float32)
        assert np.all(np.abs(got.astype(np.float64) - ref) <= np.spacing(np.abs(r32)).astype(np.float64))
        assert np.mean(got == r32) > 0.99


def test_cgemm_error_scale_invariance_and_tail_order():
    A, B = complex64_inputs(24, 18, 128, 0.5, 31)
    ref = A.astype(np.complex128) @ B.astype(np.complex128)
    C = O.cgemm(A, B, 10, PROP)
    assert np.max(np.abs(C - ref) / np.abs(ref)) < 1e-5
    C2 = O.cgemm(A * np.float32(2.0 ** 20), B * np.complex64(2.0 ** -30 * 1j), 10, PROP)
    assert np.array_equal(C2, C * np.complex64(2.0 ** -10 * 1j))
    alpha, beta = 0.5 - 2.0j, -1.25 + 0.75j
    rng = np.random.Generator(np.random.PCG64(4))
    Cin = (rng.standard_normal((24, 18)) + 1j * rng.standard_normal((24, 18))).astype(np.complex64)
    out = O.cgemm(A, B, 10, PROP, alpha=alpha, beta=beta, C_in=Cin)
    f = np.float32
    ar, ai, br, bi = f(alpha.real), f(alpha.imag), f(beta.real), f(beta.imag)
    tr = (ar * C.real - ai * C.imag) + (br * Cin.real - bi * Cin.imag)        # float32 arrays: every operation rounds to FP32
    ti = (ar * C.imag + ai * C.real) + (br * Cin.imag + bi * Cin.real)
    assert out.dtype == np.complex64 and tr.dtype == np.float32
    assert np.array_equal(out.real, tr) and np.array_equal(out.imag, ti)
