"""Pins for the oracle's scaling step (O2, O3): the three modes of computing mu, nu.

What fixes the expected values here (never the oracle itself):
  * the paper's worked example on all-ones matrices (tests/golden/fig1_*.txt),
  * the inequalities the paper derives the formulas from, evaluated in exact rational
    arithmetic: bound (16) for the revised mode, eq. (11) for the original fast
    mode, the proof chain of accurate mode, condition (1) itself,
  * closed forms on all-ones inputs where __log2f(1) = 0 makes every rounding explicit,
  * the scale-invariance statement of section 4 and its failure for Alg. 1
    (P:217-236),
  * numpy recomputation of the accurate-mode INT8 auxiliary product.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O
from exact_helpers import floor_log2, frac_sumsq, pow2, round_dir_f32

ACCU, FAST, PROP = O.MODE_ACCURATE, O.MODE_FAST, O.MODE_PROP


# ------------------------------------------------------------------ statistics (O2)
def test_row_statistics_exact_rational():
    A, B = W.wide_exponent_matrices(12, 9, 40, seed=21)
    A[3, :] = np.ldexp(1.0, -1074)                 # a row of smallest subnormals
    A[4, 0] = 5e-324
    _, _, ext = O.exponents(PROP, 14, A, B, extras=True)
    for i in range(A.shape[0]):
        row = A[i, :]
        vmax = np.abs(row).max()
        if vmax == 0:
            assert ext["SA"][i] == 0
            continue
        E = floor_log2(vmax)
        assert ext["EA"][i] == E                    # floor(log2 max), true value for subnormals
        S = 0
        for x in row:
            t = (Fraction(float(x)) / pow2(E)) ** 2 * (1 << 44)
            S += math.ceil(t)                       # reading R2: rounded-up term by term, exact integer sum
        assert int(ext["SA"][i]) == S
        # "computed with rounding-up": an upper bound of the true sum of squares ...
        assert Fraction(S, 1 << 44) * pow2(2 * E) >= frac_sumsq(row)
        # ... that exceeds it by less than k units of 2^-44 relative to the max^2
        assert Fraction(S, 1 << 44) * pow2(2 * E) < frac_sumsq(row) + len(row) * pow2(2 * E - 44)
    for j in range(B.shape[1]):
        col = B[:, j]
        if np.abs(col).max() == 0:
            continue
        assert ext["EB"][j] == floor_log2(np.abs(col).max())


# ------------------------------------------------------------------ revised fast mode (Algorithm 2)
@pytest.mark.parametrize("N,phi,seed", [(14, 0.5, 1), (8, 1.0, 2), (20, 4.0, 3), (17, 2.0, 4)])
def test_prop_mode_satisfies_and_saturates_bound16(N, phi, seed):
    A, B = W.eq15_matrices(48, 40, 96, phi, seed)
    e, f = O.exponents(PROP, N, A, B)
    P = O.constants(N)["P"]
    half = Fraction(P - 1, 2)
    loose = 0
    vecs = [(A[i, :], e[i]) for i in range(A.shape[0])] + [(B[:, j], f[j]) for j in range(B.shape[1])]
    for vec, ex in vecs:
        S = frac_sumsq(vec)
        # eq. (16)/(17):  mu_i^2 ||a_i||^2 <= (P-1)/2
        assert pow2(2 * ex) * S <= half
        # mu is "the largest power of two satisfying this bound" up to the rounding slack:
        assert pow2(2 * (ex + 2)) * S > half
        loose += pow2(2 * (ex + 1)) * S <= half
    assert loose <= 0.02 * len(vecs) + 1


@pytest.mark.parametrize("N", [8, 14, 16, 18, 20])
@pytest.mark.parametrize("logk", [7, 10, 13, 14, 16])
def test_prop_and_accu_closed_form_all_ones(N, logk):
    # all-ones, k = 2^t: sum a^2 = k, __log2f(1.0) = 0, so Algorithm 2 reads
    #   e = floor( single_down(P'_prop - t/2) - 2 u32 )
    # and accurate mode (abar = bbar = 32, cbar = 1024 k; eq. (8) with reading G3)
    #   e = 5 + floor( P'_accu - delta * (10 + t) )
    k = 1 << logk
    A, B = W.all_ones_scaled(2, 3, k, 1.0)
    c = O.constants(N)
    Pp = Fraction(float(c["Pprop"]))
    want_prop = math.floor(Pp - Fraction(logk, 2) - Fraction(1, 1 << 23))
    e, f = O.exponents(PROP, N, A, B)
    assert set(e) == {want_prop} and set(f) == {want_prop}
    want_accu = 5 + math.floor(Pp - Fraction(float(c["delta"])) * (10 + logk))
    e, f, ext = O.exponents(ACCU, N, A, B, extras=True)
    assert set(ext["rowmax"]) == {1024 * k} and set(ext["colmax"]) == {1024 * k}
    assert set(e) == {want_accu} and set(f) == {want_accu}
    # both keep A'B' = k 2^(2e) below P/2 (condition (1))
    assert k * 4 ** want_prop < c["P"] // 2 and k * 4 ** want_accu < c["P"] // 2


def test_prop_mode_scale_invariance_powers_of_two():
    # the effective bit width does not depend on alpha = 2^s; A' is unchanged.
    A, B = W.eq15_matrices(24, 20, 64, 1.0, 9)
    N = 16
    e0, f0, x0 = O.exponents(PROP, N, A, B, extras=True)
    A0 = O.truncate(0, A, e0)
    R0 = O.residues(1, N, B, f0)
    for s in (-500, -3, 7, 500):
        c = 2.0 ** s
        e1, f1, x1 = O.exponents(PROP, N, A * c, B * c, extras=True)
        assert np.array_equal(e1, e0 - s) and np.array_equal(f1, f0 - s)
        assert np.array_equal(x1["EA"], x0["EA"] + s)
        assert np.array_equal(e1 + x1["EA"], e0 + x0["EA"])          # effective bit width
        assert np.array_equal(O.truncate(0, A * c, e1), A0)
        assert np.array_equal(O.residues(1, N, B * c, f1), R0)


def test_prop_mode_scale_non_power_of_two_moves_width_by_at_most_one():
    A, B = W.eq15_matrices(32, 8, 128, 1.0, 10)
    e0, _, x0 = O.exponents(PROP, 14, A, B, extras=True)
    for c in (1e100, 1e-100, 3.0):
        e1, _, x1 = O.exponents(PROP, 14, A * c, B * c, extras=True)
        d = (e1 + x1["EA"]) - (e0 + x0["EA"])
        assert np.abs(d).max() <= 1


# ------------------------------------------------------------------ original fast mode (Algorithm 1)
def test_fast_mode_paper_worked_example(golden):
    g = golden("fig1_allones_fastmode.txt")
    N = int(g["N"])
    thr = int(g["violation_iff_s_le"])
    c = O.constants(N)
    P = c["P"]
    plateau = math.floor(Fraction(float(c["Pfast"])) - 1)       # floor(P'_fast - 1)
    for k in (int(x) for x in g["k_values"].split(",")):
        for s in range(int(g["s_min"]), int(g["s_max"]) + 1):
            alpha = 2.0 ** s
            A, B = W.all_ones_scaled(2, 2, k, alpha)
            e, f = O.exponents(FAST, N, A, B)
            Ap = O.pairs_to_ints(O.truncate(0, A, e))
            Bp = O.pairs_to_ints(O.truncate(1, B, f))
            z = sum(int(Ap[0, h]) * int(Bp[0, h]) for h in range(k))
            # P:257 "exceeds the CRT recovery threshold P/2 in the region alpha <= 2^-2"
            assert (z > P // 2) == (s <= thr), (k, s)
            if alpha * alpha * k <= 1:                           # alpha <= k^(-1/2)
                assert set(Ap.ravel()) == {1 << plateau} and set(Bp.ravel()) == {1 << plateau}
                assert z == k * 4 ** plateau
            # the revised mode on the same inputs never violates and ignores alpha
            e2, f2 = O.exponents(PROP, N, A, B)
            assert k * 4 ** (int(e2[0]) + s) < P // 2
            assert int(e2[0]) + s == int(O.exponents(PROP, N, *W.all_ones_scaled(2, 2, k, 1.0))[0][0])


@pytest.mark.parametrize("N,phi,seed", [(14, 0.5, 5), (20, 1.0, 6), (10, 2.0, 7)])
def test_fast_mode_eq11_in_exact_arithmetic(N, phi, seed):
    # eq. (11): effective width - 1 = floor(P'_fast - max(1, delta log2~(sum a^2))).
    # With 2^(2 P'_fast) <= (P-1)/8:   in the regime sum a^2 >= 4 the scaled row obeys
    # (2^(e+E))^2 sum a^2 <= (P-1)/8, and does so tightly; below it the width is the plateau.
    A, B = W.eq15_matrices(40, 8, 512, phi, seed)
    A *= 8.0                                                     # put rows into the "t > 1" regime
    c = O.constants(N)
    P = c["P"]
    e, _, ext = O.exponents(FAST, N, A, B, extras=True)
    loose = 0
    for i in range(A.shape[0]):
        S = frac_sumsq(A[i, :])
        assert S >= 4
        w = int(e[i]) + int(ext["EA"][i])
        assert pow2(2 * w) * S <= Fraction(P - 1, 8)
        assert pow2(2 * (w + 2)) * S > Fraction(P - 1, 8)
        loose += pow2(2 * (w + 1)) * S <= Fraction(P - 1, 8)
    assert loose <= 2
    # tiny inputs: plateau floor(P'_fast - 1)
    e, _, ext = O.exponents(FAST, N, A * 2.0 ** -40, B, extras=True)
    assert set(e + ext["EA"]) == {math.floor(Fraction(float(c["Pfast"])) - 1)}


def test_fast_mode_is_not_scale_invariant_but_prop_is():
    # eq. (13): above the plateau one bit is lost per doubling of alpha.
    A, B = W.eq15_matrices(16, 4, 256, 0.5, 8)
    A *= 16.0
    e0, _, x0 = O.exponents(FAST, 18, A, B, extras=True)
    w0 = e0 + x0["EA"]
    for s in (1, 2, 5, 40):
        e1, _, x1 = O.exponents(FAST, 18, A * 2.0 ** s, B, extras=True)
        assert np.array_equal(e1 + x1["EA"], w0 - s)
        e2, _, x2 = O.exponents(PROP, 18, A * 2.0 ** s, B, extras=True)
        e3, _, x3 = O.exponents(PROP, 18, A, B, extras=True)
        assert np.array_equal(e2 + x2["EA"], e3 + x3["EA"])


# ------------------------------------------------------------------ accurate mode
@pytest.mark.parametrize("N,phi,seed", [(14, 0.5, 11), (20, 4.0, 12), (9, 1.0, 13)])
def test_accurate_mode_auxiliary_product_and_bound(N, phi, seed):
    A, B = W.eq15_matrices(36, 28, 80, phi, seed)
    e, f, ext = O.exponents(ACCU, N, A, B, extras=True)
    EA = np.array([floor_log2(np.abs(A[i, :]).max()) for i in range(A.shape[0])])
    EB = np.array([floor_log2(np.abs(B[:, j]).max()) for j in range(B.shape[1])])
    assert np.array_equal(ext["EA"], EA) and np.array_equal(ext["EB"], EB)
    # Abar = ceil(mu' |a|), mu' = 2^(5 - E): exact in FP64 for these magnitudes
    Ab = np.ceil(np.abs(A) * np.exp2(5.0 - EA)[:, None]).astype(np.int64)
    Bb = np.ceil(np.abs(B) * np.exp2(5.0 - EB)[None, :]).astype(np.int64)
    assert Ab.max() <= 64 and Bb.max() <= 64 and Ab.max() >= 32
    Cb = Ab @ Bb
    assert np.array_equal(ext["rowmax"], Cb.max(axis=1))
    assert np.array_equal(ext["colmax"], Cb.max(axis=0))
    P = O.constants(N)["P"]
    # proof chain P:159-163 with reading G3: (mu_i/mu'_i)^2 max_j cbar_ij <= (P-1)/2, tightly
    for ex, E, M in [(e[i], EA[i], Cb[i, :].max()) for i in range(len(e))] + \
                    [(f[j], EB[j], Cb[:, j].max()) for j in range(len(f))]:
        r = int(ex) - (5 - int(E))
        assert pow2(2 * r) * int(M) <= Fraction(P - 1, 2)
        assert pow2(2 * (r + 2)) * int(M) > Fraction(P - 1, 2)
    # and therefore condition (1), exactly
    s = O.stages(A, B, N, ACCU, want_exact=True)
    assert s["counts"] == dict(violations=0, wrong=0)


def test_zero_rows_and_columns_get_exponent_zero():
    A, B = W.wide_exponent_matrices(10, 9, 32, seed=3)
    for mode in (ACCU, FAST, PROP):
        e, f = O.exponents(mode, 14, A, B)
        assert e[10 // 2] == 0 and f[9 // 3] == 0               # reading R4
        RA = O.residues(0, 14, A, e)
        assert not RA[:, 10 // 2, :].any()


# ------------------------------------------------------------------ condition (1) on random data
@pytest.mark.parametrize("mode", [ACCU, PROP])
@pytest.mark.parametrize("N,phi", [(8, 0.5), (14, 1.0), (16, 4.0), (20, 2.0)])
def test_condition_1_always_holds_for_accu_and_prop(mode, N, phi):
    # P:358 / P:440 (revised mode), P:159-163 (accurate mode)
    A, B = W.eq15_matrices(24, 24, 200, phi, 100 + N)
    s = O.stages(A, B, N, mode, want_exact=True)
    assert s["counts"] == dict(violations=0, wrong=0)


def test_condition_1_wide_exponent_inputs_prop():
    A, B = W.wide_exponent_matrices(16, 16, 64, seed=77)
    s = O.stages(A, B, 20, PROP, want_exact=True)
    assert s["counts"] == dict(violations=0, wrong=0)


def test_prop_mode_2u32_term_on_boundary_rows():
    # Algorithm 2 line 2: t = single_up(0.5 * __log2f(a_norm / 2^s) + 2 u32).  The 2 u32
    # term only shows when w - 0.5 L sits within 2^-23 above an integer; build such rows (one non-zero
    # entry v in [1,2), so E = 0 and a_norm = v^2) and evaluate the algorithm's three lines in exact
    # rational arithmetic with the roundings it prescribes.
    bits = np.arange(0x3F800000, 0x40000000, dtype=np.uint32)
    xs = bits.view(np.float32)
    Ls = np.log2(xs.astype(np.float64)).astype(np.float32)       # = LOG2F, pinned in test_oracle_log2f.py
    hits = 0
    for N in range(2, 21):
        Pp = Fraction(float(O.constants(N)["Pprop"]))
        for shat in (0, 1):
            w = round_dir_f32(Pp - Fraction(shat, 2), up=False)
            fr = Fraction(float(w)) - math.floor(Fraction(float(w)))
            lo, hi = float(2 * fr) - 2.0 ** -22, float(2 * fr)
            idx = np.nonzero((Ls.astype(np.float64) > lo) & (Ls.astype(np.float64) <= hi))[0]
            for t in idx[:1]:
                x0, L = float(xs[t]), Fraction(float(Ls[t]))
                v = math.sqrt(x0 * 2.0 ** shat * (1 - 2.0 ** -25))
                A = np.zeros((1, 4), order="F")
                A[0, 1] = -v
                B = np.ones((4, 1), order="F")
                e, _, ext = O.exponents(PROP, N, A, B, extras=True)
                S = math.ceil(Fraction(v) ** 2 * (1 << 44))
                assert int(ext["SA"][0]) == S and ext["EA"][0] == 0
                F = round_dir_f32(Fraction(S), up=True)
                assert Fraction(float(F)) == Fraction(x0) * pow2(44 + shat)      # the row hits the target x0
                tt = round_dir_f32(L / 2 + Fraction(1, 1 << 23), up=True)
                d = round_dir_f32(Fraction(float(w)) - Fraction(float(tt)), up=False)
                want = math.floor(Fraction(float(d)))
                without = math.floor(Fraction(float(round_dir_f32(Fraction(float(w)) - L / 2, up=False))))
                assert without == want + 1                                        # the case is sensitive
                assert int(e[0]) == want
                hits += 1
    assert hits >= 10


# --------------------------------------------------------------------------------------------- k > 2^17
def _sq_shift(k):
    lg = max(0, (k - 1).bit_length())
    extra = max(0, lg - 17)
    return 44 - 2 * ((extra + 1) // 2)


@pytest.mark.parametrize("k", [(1 << 17) + 5, (1 << 18), (1 << 19) + 1])
def test_long_k_row_statistics_exact_integers(k):
    # reading R2b: beyond k = 2^17 the fixed-point position of the rounded-up sum drops by 2 per factor 4 of k
    import math
    rng = np.random.Generator(np.random.PCG64(k))
    A = np.asfortranarray(((rng.random((1, k)) - 0.5) * np.exp(rng.standard_normal((1, k)))))
    Bm = np.asfortranarray(np.ones((k, 1)))
    _, _, ext = O.exponents(PROP, 14, A, Bm, extras=True)
    SQ = _sq_shift(k)
    assert SQ == {131077: 42, 262144: 42, 524289: 40}[k]
    row = A[0]
    E = floor_log2(np.max(np.abs(row)))
    S = 0
    for x in row.tolist():                      # exact: |x| = M 2^q, term = ceil(M^2 2^(2(q-E)+SQ))
        mant, ex = math.frexp(abs(x))
        M, q = int(mant * (1 << 53)), ex - 53
        r = -(2 * (q - E) + SQ)
        assert r > 0
        S += (M * M + (1 << r) - 1) >> r
    assert int(ext["SA"][0]) == S and S < 2 ** 63
    assert Fraction(S, 1 << SQ) * pow2(2 * E) >= sum(Fraction(x) ** 2 for x in row[:2000].tolist())


@pytest.mark.parametrize("N,t", [(14, 18), (16, 19), (20, 20)])
def test_long_k_all_ones_closed_form(N, t):
    # all-ones, k = 2^t: the normalised sum is exactly k, LOG2F(1) = 0, so Algorithm 2 gives
    # e = floor(single_down(P'_prop - t/2) - 2^-23) whatever the fixed-point position is;
    # P'_prop - t/2 is exact in FP32 here (same binade or coarser) and its fraction is far from 0 and 2^-23
    k = 1 << t
    A, Bm = W.all_ones_scaled(2, 2, k, 1.0)
    e, f = O.exponents(PROP, N, A, Bm)
    c = O.constants(N)
    want = int(np.floor(float(c["Pprop"]) - 0.5 * t - 2.0 ** -23))
    assert e[0] == want == f[0]
    assert 2 * k * (1 << (2 * want)) < c["P"]                    # condition (1): k 2^(2e) < P / 2


def test_long_k_condition_1_and_recovery_random():
    k = (1 << 18) + 37
    A, Bm = W.eq15_matrices(3, 2, k, 1.0, 77)
    st = O.stages(A, Bm, 16, PROP, want_exact=True)
    assert st["counts"]["violations"] == 0 and st["counts"]["wrong"] == 0
    assert np.array_equal(st["Cpp"], st["Z"])
