"""Pins for the oracle's last steps (O9, O10) and for the whole path.

Expected values: textbook special cases (integer matrices, identity, all-ones), exact rational
arithmetic with CPython's correctly rounded int/Fraction -> float conversion, and the paper's
own statements about accuracy (Fig. 2 breakdown thresholds P:293, prop ~ accu P:383).
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O
from exact_helpers import pow2, trunc_scaled

ACCU, FAST, PROP = O.MODE_ACCURATE, O.MODE_FAST, O.MODE_PROP


def max_rel_err(Cm, A, B):
    hi, lo = O.dd_reference(A, B)
    nz = hi != 0
    return float(np.max(np.abs((Cm - hi) - lo)[nz] / np.abs(hi[nz])))


def test_dd_reference_against_exact_rationals():
    A, B = W.eq15_matrices(5, 4, 33, 2.0, 2)
    hi, lo = O.dd_reference(A, B)
    for i in range(5):
        for j in range(4):
            x = sum(Fraction(float(A[i, h])) * Fraction(float(B[h, j])) for h in range(33))
            got = Fraction(float(hi[i, j])) + Fraction(float(lo[i, j]))
            assert abs(got - x) <= abs(x) * Fraction(1, 1 << 95)
            assert hi[i, j] == float(x)                    # hi is the correctly rounded double


@pytest.mark.parametrize("mode", [ACCU, FAST, PROP])
def test_small_integer_matrices_give_the_exact_integer_product(mode):
    A, B = W.small_integer_matrices(17, 13, 64, bound=8, seed=4)
    want = A.astype(np.int64) @ B.astype(np.int64)
    got = O.dgemm(A, B, 14, mode)
    assert np.array_equal(got, want.astype(np.float64))


@pytest.mark.parametrize("mode", [ACCU, PROP])
def test_identity_times_b_is_truncation_of_b(mode):
    # A = I: c_ij = trunc(nu_j b_ij) / nu_j exactly (Step 2 and Step 4)
    n, k = 9, 12
    _, B = W.eq15_matrices(k, n, k, 1.0, 6)
    A = np.asfortranarray(np.eye(k))
    got, e, f = O.dgemm(A, B, 12, mode, return_exponents=True)
    for i in range(k):
        for j in range(n):
            want = Fraction(trunc_scaled(B[i, j], int(f[j]))) / pow2(int(f[j]))
            assert Fraction(float(got[i, j])) == want


@pytest.mark.parametrize("s", [-10, -3, 0, 4, 10])
@pytest.mark.parametrize("k", [256, 1024])
def test_all_ones_times_alpha_is_exact_for_prop_and_accu(s, k):
    # exact arithmetic gives error 0 on this input; the revised and accurate modes reproduce it
    alpha = 2.0 ** s
    A, B = W.all_ones_scaled(3, 2, k, alpha)
    for mode in (PROP, ACCU):
        assert np.all(O.dgemm(A, B, 20, mode) == k * alpha * alpha)


def test_final_c_is_rn_of_exact_product_then_exact_scaling():
    # reading R8: C = RN_64(C'') 2^-(e_i+f_j); C'' = A'B' (pinned in test_oracle_integer_stages.py)
    A, B = W.eq15_matrices(8, 7, 60, 4.0, 12)
    for mode, N in ((PROP, 20), (ACCU, 16), (PROP, 9)):
        s = O.stages(A, B, N, mode, want_exact=True)
        Ap = O.pairs_to_ints(s["Ap"])
        Bp = O.pairs_to_ints(s["Bp"])
        for i in range(8):
            for j in range(7):
                z = sum(int(Ap[i, h]) * int(Bp[j, h]) for h in range(60))
                want = float(Fraction(z) / pow2(int(s["e"][i]) + int(s["f"][j])))
                assert s["C"][i, j] == want
    assert np.array_equal(O.dgemm(A, B, 9, PROP), s["C"])   # the one-call entry gives the same C


def test_subnormal_and_overflowing_results_round_once():
    A = np.asfortranarray(np.array([[2.0 ** -600, 3 * 2.0 ** -610], [2.0 ** 600, 2.0 ** 590]]))
    B = np.asfortranarray(np.array([[1.5 * 2.0 ** -470, 2.0 ** 500], [2.0 ** -466 + 2.0 ** -500, 2.0 ** 510]]))
    got, e, f = O.dgemm(A, B, 20, PROP, return_exponents=True)
    for i in range(2):
        for j in range(2):
            z = sum(trunc_scaled(A[i, h], int(e[i])) * trunc_scaled(B[h, j], int(f[j])) for h in range(2))
            x = Fraction(z) / pow2(int(e[i]) + int(f[j]))
            try:
                want = float(x)
            except OverflowError:
                want = math.inf
            assert got[i, j] == want
    assert 0 < got[0, 0] < 2.0 ** -1022 and got[1, 1] == math.inf


def test_alpha_beta_semantics():
    # reading R9: t = alpha * c (RN); out = t if beta == 0 else fma(beta, C_in, t); beta == 0 ignores C_in
    A, B = W.eq15_matrices(6, 5, 32, 1.0, 14)
    c = O.dgemm(A, B, 14, PROP)
    Cin = np.asfortranarray(np.random.Generator(np.random.PCG64(1)).standard_normal((6, 5)))
    alpha, beta = 0.7, -1.3
    got = O.dgemm(A, B, 14, PROP, alpha=alpha, beta=beta, C_in=Cin)
    for i in range(6):
        for j in range(5):
            t = alpha * c[i, j]
            want = float(Fraction(beta) * Fraction(float(Cin[i, j])) + Fraction(t))
            assert got[i, j] == want
    nanC = np.full((6, 5), np.nan, order="F")
    assert np.array_equal(O.dgemm(A, B, 14, PROP, alpha=2.0, beta=0.0, C_in=nanC), 2.0 * c)


def test_scale_invariance_of_the_result():
    # P:354-358 + reading R12: for c = 2^s the revised mode gives C(cA, cB) = c^2 C(A, B) exactly;
    # the original fast mode does not keep its accuracy.
    A, B = W.eq15_matrices(16, 16, 128, 1.0, 31)
    c0 = O.dgemm(A, B, 15, PROP)
    for s in (-480, -7, 9, 480):
        c = 2.0 ** s
        assert np.array_equal(O.dgemm(A * c, B * c, 15, PROP), c0 * c * c)
    e_small = max_rel_err(O.dgemm(A, B, 15, FAST), A, B)
    e_big = max_rel_err(O.dgemm(A * 2.0 ** 12, B * 2.0 ** 12, 15, FAST), A * 2.0 ** 12, B * 2.0 ** 12)
    assert e_big > 100 * e_small


def test_accuracy_trends_of_the_paper():
    # prop keeps accuracy comparable to accu for every phi; fast degrades as phi grows.
    # errors decrease as N increases.
    errs = {}
    for phi in (0.5, 4.0):
        A, B = W.eq15_matrices(48, 48, 256, phi, 50)
        for mode in (ACCU, FAST, PROP):
            errs[(phi, mode)] = max_rel_err(O.dgemm(A, B, 14, mode), A, B)
    assert errs[(0.5, PROP)] < 1e-10 and errs[(0.5, ACCU)] < 1e-10 and errs[(0.5, FAST)] < 1e-9
    for phi in (0.5, 4.0):
        assert errs[(phi, PROP)] < 16 * errs[(phi, ACCU)]
    assert errs[(4.0, FAST)] > 50 * errs[(4.0, PROP)]
    A, B = W.eq15_matrices(32, 32, 256, 1.0, 51)
    e10, e14, e18 = (max_rel_err(O.dgemm(A, B, N, PROP), A, B) for N in (10, 14, 18))
    assert e10 > 1e3 * e14 and e14 > 1e3 * e18 and e18 < 1e-14


def test_fast_mode_breakdown_thresholds_of_fig2(golden):
    # phi = 0.5, N = 20: max rel err ~ 1 for alpha <= 2^-3 (k = 1024, m = n = 1024) and for
    # alpha <= 2^-5 (k = 16384), fine above; accurate and revised modes are unaffected.
    # The breakdown is a max over ~10^6 entries (an entry of A'B' beyond P/2), so the search for
    # violating entries uses the oracle's Algorithm-1 exponents with an FP64 matmul of the scaled matrices
    # (relative accuracy 1e-13 is ample for a > P/2 test); the full oracle path then runs on an 8x8 slab
    # around the worst entry.
    g = golden("fig2_fastmode_breakdown.txt")
    N, phi = int(g["N"]), float(g["phi"])
    half_P = float(O.constants(N)["P"]) / 2
    for k, mn, thr in ((1024, 1024, int(g["breakdown_s_le_k1024"])), (16384, 2048, int(g["breakdown_s_le_k16384"]))):
        A, B = W.eq15_matrices(mn, mn, k, phi, 60 + k)
        for s, broken in ((thr - 1, True), (thr, True), (thr + 1, False), (thr + 3, False)):
            c = 2.0 ** s
            e, f = O.exponents(FAST, N, A * c, B * c)
            Z = (np.trunc(A * c * np.exp2(e.astype(np.float64))[:, None])) @ (np.trunc(B * c * np.exp2(f.astype(np.float64))[None, :]))
            worst = np.unravel_index(np.argmax(np.abs(Z)), Z.shape)
            assert (abs(Z[worst]) > half_P * (1 + 1e-9)) == broken, (k, s)
            assert abs(abs(Z[worst]) / half_P - 1) > 1e-6                       # not a borderline call
            i0, j0 = (worst[0] // 8) * 8, (worst[1] // 8) * 8
            As, Bs = A[i0:i0 + 8, :] * c, B[:, j0:j0 + 8] * c
            err = max_rel_err(O.dgemm(As, Bs, N, FAST), As, Bs)
            assert (err > 1e-2) == broken, (k, s, err)
            if broken:
                assert max_rel_err(O.dgemm(As, Bs, N, PROP), As, Bs) < 1e-14
                assert max_rel_err(O.dgemm(As, Bs, N, ACCU), As, Bs) < 1e-14
