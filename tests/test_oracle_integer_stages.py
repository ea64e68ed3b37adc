"""Pins for the oracle's integer stages: truncation (O4), residues (O5), per-modulus
products (O6), CRT recovery (O7) and the exact product / condition (1) check (O8).

Expected values come from Python's arbitrary-precision integers and exact rationals
(the plain definitions: trunc, mod, the sum of products, Theorem 1), never from the oracle.
"""
import itertools
import random

import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O
from exact_helpers import sym_mod, trunc_scaled

ACCU, FAST, PROP = O.MODE_ACCURATE, O.MODE_FAST, O.MODE_PROP


def test_truncation_is_exact_trunc_of_scaled_value():
    # a' = trunc(mu_i a), against exact rationals, over the whole FP64 exponent range
    A, B = W.wide_exponent_matrices(14, 10, 48, seed=5)
    A[1, :] = A[0, :] * 2.0 ** -30          # rows whose entries are mostly shifted out
    for mode, N in ((PROP, 20), (ACCU, 20), (FAST, 9)):
        e, f = O.exponents(mode, N, A, B)
        Ap = O.pairs_to_ints(O.truncate(0, A, e))
        Bp = O.pairs_to_ints(O.truncate(1, B, f))
        for i in range(A.shape[0]):
            for h in range(A.shape[1]):
                assert int(Ap[i, h]) == trunc_scaled(A[i, h], int(e[i]))
        for j in range(B.shape[1]):
            for h in range(B.shape[0]):
                assert int(Bp[j, h]) == trunc_scaled(B[h, j], int(f[j]))
    # widths stay below floor(P') + 1 (+6 for accurate mode): the oracle's int128 is wide enough
    assert max(abs(int(v)) for v in Ap.ravel()).bit_length() <= 84


def test_truncation_small_exponents_and_signs():
    X = np.asfortranarray(np.array([[1.5, -1.5, 0.75, -0.75, 3.999, -3.999, 0.0, -0.0, 2.0 ** -60, 1e-320]]))
    for ex in (-2, -1, 0, 1, 5, 52, 60):
        got = O.pairs_to_ints(O.truncate(0, X, np.array([ex], np.int32)))
        for h in range(X.shape[1]):
            assert int(got[0, h]) == trunc_scaled(X[0, h], ex)


@pytest.mark.parametrize("N", [2, 9, 14, 20])
def test_residues_are_symmetric_representatives(N):
    A, B = W.eq15_matrices(10, 8, 96, 2.0, 40 + N)
    p = O.constants(N)["p"]
    e, f = O.exponents(PROP, N, A, B)
    for op, X, ex in ((0, A, e), (1, B, f)):
        R = O.residues(op, N, X, ex)
        T = O.pairs_to_ints(O.truncate(op, X, ex))
        assert R.dtype == np.int8
        for l in range(N):
            for r in range(T.shape[0]):
                for h in range(T.shape[1]):
                    assert int(R[l, r, h]) == sym_mod(int(T[r, h]), p[l])      # rmod, P:70 (reading R5)
            if p[l] % 2:
                assert R[l].min() >= -(p[l] - 1) // 2 and R[l].max() <= (p[l] - 1) // 2
    # negating the input negates the residues of odd moduli
    Rn = O.residues(0, N, -A, e)
    Rp = O.residues(0, N, A, e)
    for l in range(N):
        if p[l] % 2:
            assert np.array_equal(Rn[l], -Rp[l])


def test_residue_of_256_is_low_byte():
    X = np.asfortranarray(np.array([[128.0, -128.0, 127.0, -129.0, 384.0, 255.0, 256.0, -1.0]]))
    R = O.residues(0, 2, X, np.array([0], np.int32))
    assert list(R[0, 0]) == [-128, -128, 127, 127, -128, -1, 0, -1]            # two's-complement low byte
    assert list(R[1, 0]) == [sym_mod(int(v), 255) for v in X[0]]


@pytest.mark.parametrize("N", [3, 14, 20])
def test_products_match_integer_matmul_mod_p(N):
    rng = np.random.Generator(np.random.PCG64(N))
    m, n, k = 13, 11, 300
    p = O.constants(N)["p"]
    RA = np.stack([rng.integers(-(q // 2), (q - 1) // 2 + 1, size=(m, k)) for q in p]).astype(np.int8)
    RB = np.stack([rng.integers(-(q // 2), (q - 1) // 2 + 1, size=(n, k)) for q in p]).astype(np.int8)
    U, maxR = O.products(N, RA, RB)
    mx = 0
    for l in range(N):
        Rl = RA[l].astype(np.int64) @ RB[l].astype(np.int64).T                 # [m][n]
        mx = max(mx, int(np.abs(Rl).max()))
        assert np.array_equal(U[l], (Rl % p[l]).T.astype(np.uint8))            # U[l][j][i], in [0, p)
    assert maxR == mx


def test_int32_headroom_bound_k_2pow17():
    # k <= 2^17 keeps the INT32 accumulator from overflowing -- with |r| <= 127 for the odd
    # moduli; p = 256 may reach 128 * 128 * 2^17 = 2^31, harmless because 256 | 2^32 (reading R6).
    k = 1 << 17
    RA = np.full((2, 1, k), -128, np.int8)
    RB = np.full((2, 1, k), -128, np.int8)
    RA[1] = 127
    RB[1] = 127
    U, maxR = O.products(2, RA, RB)
    assert maxR == 2 ** 31
    assert U[0, 0, 0] == (2 ** 31) % 256 == 0
    assert U[1, 0, 0] == (127 * 127 * k) % 255
    assert 127 * 127 * k < 2 ** 31


def _crt_of_int(N, z):
    p = O.constants(N)["p"]
    U = np.array([z % q for q in p], np.uint8).reshape(N, 1, 1)
    return O.words_to_int(O.crt(N, U)[0, 0])


def test_crt_exhaustive_two_moduli():
    # Theorem 1 + eq. (3): every integer of [-P/2, P/2) is recovered from its residues. N = 2: all of them.
    N = 2
    P = O.constants(N)["P"]
    p = O.constants(N)["p"]
    zs = np.arange(-P // 2, P // 2)
    U = np.stack([(zs % q).astype(np.uint8) for q in p]).reshape(N, 1, P)
    got = O.words_array_to_ints(O.crt(N, U))[0]
    assert [int(g) for g in got] == [int(z) for z in zs]


@pytest.mark.parametrize("N", range(3, 21))
def test_crt_random_and_boundary_values(N):
    P = O.constants(N)["P"]
    rng = random.Random(N)
    zs = [0, 1, -1, P // 2 - 1, -(P // 2), P // 2 - 2, -(P // 2) + 1]
    zs += [rng.randrange(-(P // 2), P // 2) for _ in range(60)]
    zs += [rng.randrange(-(1 << b), 1 << b) for b in (1, 8, 30, 60) if (1 << b) < P // 2]
    for z in zs:
        assert _crt_of_int(N, z) == z
    # outside the range the result is the representative of z mod P in [-P/2, P/2) (reading R7)
    for z in (P // 2, P // 2 + 5, -(P // 2) - 1, 3 * P + 7):
        want = ((z + P // 2) % P) - P // 2
        assert _crt_of_int(N, z) == want


def test_brute_force_tiny_integer_matrices():
    # north_star: "a brute-force check on tiny inputs that the CRT recovers [A'B'] whenever |A'B'| < P/2".
    # Enumerate ALL 2x2 integer matrices with entries in {-2..2}; with integer inputs and exponents forced
    # to 0 the scaled matrices are the inputs themselves.
    vals = (-2, -1, 0, 1, 2)
    mats = [np.array(t, dtype=np.float64).reshape(2, 2) for t in itertools.product(vals, repeat=4)]
    z = np.zeros(2, np.int32)
    for N in (2, 3, 6):
        for Am in mats[::7]:
            RA = O.residues(0, N, np.asfortranarray(Am), z)
            for Bm in mats[::11]:
                RB = O.residues(1, N, np.asfortranarray(Bm), z)
                U, _ = O.products(N, RA, RB)
                got = O.words_array_to_ints(O.crt(N, U))           # [n][m]
                want = Am.astype(np.int64) @ Bm.astype(np.int64)
                assert np.array_equal(got.T.astype(np.int64), want)


@pytest.mark.parametrize("mode,N,phi", [(PROP, 6, 0.5), (PROP, 14, 1.0), (ACCU, 17, 4.0), (PROP, 20, 4.0), (FAST, 12, 1.0)])
def test_crt_recovers_exact_product_python_integers(mode, N, phi):
    A, B = W.eq15_matrices(9, 7, 50, phi, 300 + N)
    s = O.stages(A, B, N, mode, want_exact=True)
    Ap = O.pairs_to_ints(s["Ap"])
    Bp = O.pairs_to_ints(s["Bp"])
    P = O.constants(N)["P"]
    Cpp = O.words_array_to_ints(s["Cpp"])
    Z = O.words_array_to_ints(s["Z"])
    Za = O.words_array_to_ints(s["Zabs"])
    for i in range(A.shape[0]):
        for j in range(B.shape[1]):
            z = sum(int(Ap[i, h]) * int(Bp[j, h]) for h in range(A.shape[1]))
            za = sum(abs(int(Ap[i, h]) * int(Bp[j, h])) for h in range(A.shape[1]))
            assert int(Z[j, i]) == z and int(Za[j, i]) == za          # the oracle's 256-bit product
            assert 2 * za < P                                         # condition (1)
            assert int(Cpp[j, i]) == z                                # eq. (3) recovers A'B'
    assert s["counts"] == dict(violations=0, wrong=0)


def test_fast_mode_violation_is_detected_and_congruent():
    # all-ones, alpha = 2^-4, N = 20 (inside the paper's failure region): C'' != A'B' but congruent.
    N, k = 20, 1024
    A, B = W.all_ones_scaled(3, 2, k, 2.0 ** -4)
    s = O.stages(A, B, N, FAST, want_exact=True)
    P = O.constants(N)["P"]
    Cpp = O.words_array_to_ints(s["Cpp"])
    Z = O.words_array_to_ints(s["Z"])
    assert s["counts"] == dict(violations=6, wrong=6)
    for a, b in zip(Cpp.ravel(), Z.ravel()):
        assert int(a) != int(b) and (int(a) - int(b)) % P == 0 and -P // 2 <= int(a) < P // 2


def test_recovered_integer_is_independent_of_moduli_count():
    # reading R14: with the exponents fixed, C'' = A'B' does not depend on N while (1) holds
    A, B = W.eq15_matrices(6, 5, 40, 1.0, 17)
    e, f = O.exponents(PROP, 14, A, B)
    outs = []
    for N in (14, 15, 18):
        U, _ = O.products(N, O.residues(0, N, A, e), O.residues(1, N, B, f))
        outs.append(O.words_array_to_ints(O.crt(N, U)))
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
