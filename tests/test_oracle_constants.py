"""Pins for the oracle's constants (O1) and FP32 / wide-integer primitives.

Nothing here compares the oracle with itself: eq. (14) comes from the paper's text, the
CRT identities from Theorem 1, the P' constants from a 400-bit mpmath evaluation
of the paper's formulas, the FP32 directed
operations and the integer -> double rounding from exact rational arithmetic.
"""
import math
import random
from fractions import Fraction
from math import gcd

import numpy as np
import pytest
from mpmath import mp, mpf, log

from oracle import ozaki2_oracle as O
from exact_helpers import round_dir_f32 as _round_dir


def _moduli(golden):
    return [int(x) for x in golden("eq14_moduli.txt")["moduli"].split(",")]


def test_moduli_are_eq14_prefix(golden):
    paper = _moduli(golden)
    assert len(paper) == 20
    for N in range(2, 21):
        assert O.constants(N)["p"] == paper[:N]


def test_moduli_greedy_largest_pairwise_coprime(golden):
    # BASELINE.json configs[0]: "largest pairwise-coprime <= 256"
    g = []
    for c in range(256, 1, -1):
        if all(gcd(c, x) == 1 for x in g):
            g.append(c)
        if len(g) == 20:
            break
    assert g == _moduli(golden)


@pytest.mark.parametrize("N", range(2, 21))
def test_crt_identities(N):
    c = O.constants(N)
    p, P = c["p"], c["P"]
    assert P == math.prod(p)
    for l in range(N):
        Pl = P // p[l]
        assert (Pl * c["q"][l]) % p[l] == 1            # q_l = P_l^{-1} mod p_l   (Step 1)
        assert c["w"][l] == Pl * c["q"][l]
        assert c["w"][l] % p[l] == 1
        for j in range(N):
            if j != l:
                assert c["w"][l] % p[j] == 0
    assert sum(c["w"]) % P == 1
    # Theorem 1 on random x
    rng = random.Random(N)
    for _ in range(50):
        x = rng.randrange(-P // 2, P // 2)
        assert sum(c["w"][l] * (x % p[l]) for l in range(N)) % P == x % P


def _f32_down(x):
    f = np.float32(float(x))
    if mpf(float(f)) > x:
        f = np.nextafter(f, np.float32(-np.inf))
    return np.float32(f)


def _f32_up(x):
    f = np.float32(float(x))
    if mpf(float(f)) < x:
        f = np.nextafter(f, np.float32(np.inf))
    return np.float32(f)


@pytest.mark.parametrize("N", range(2, 21))
def test_p_prime_constants_mpmath(N):
    mp.prec = 400
    c = O.constants(N)
    l2 = log(mpf(c["P"] - 1), 2)
    assert c["Pprop"] == _f32_down(l2 / 2 - mpf("0.5"))      # P:326-328 (= P'_accu)
    assert c["Pfast"] == _f32_down(l2 / 2 - mpf("1.5"))
    assert float(c["Pfast"]) == float(c["Pprop"]) - 1.0
    u32 = mpf(2) ** -24
    assert c["delta"] == _f32_up(mpf("0.5") / (1 - 4 * u32))  # eq. (6)
    assert float(c["delta"]) == float.fromhex("0x1.000006p-1")


def test_p_prime_spot_values():
    # hex floats of SURVEY Appendix A rows (400-bit mpmath at survey time), as a second witness
    assert float(O.constants(14)["Pprop"]) == float.fromhex("0x1.b4a4fep+5")
    assert float(O.constants(20)["Pprop"]) == float.fromhex("0x1.34be22p+6")
    assert float(O.constants(20)["Pfast"]) == float.fromhex("0x1.30be22p+6")
    assert O.constants(14)["P"] == 1451455329416086687492492043070720
    assert O.constants(20)["P"] == 59079700598002655956659983298716520937586883840


# ------------------------------------------------------------------ FP32 directed operations
def _rand_f32(rng, lo_exp=-30, hi_exp=12):
    m = rng.random() + 1.0
    v = np.float32(m * 2.0 ** rng.randrange(lo_exp, hi_exp))
    return np.float32(-v if rng.random() < 0.3 else v)


def test_f32_directed_ops_against_exact_rationals():
    L = O.lib()
    rng = random.Random(7)
    for _ in range(3000):
        a, b, c = _rand_f32(rng), _rand_f32(rng), _rand_f32(rng)
        fa, fb, fc = Fraction(float(a)), Fraction(float(b)), Fraction(float(c))
        for up in (0, 1):
            assert np.float32(L.oz2o_f32_add(a, b, up)) == _round_dir(fa + fb, bool(up))
            assert np.float32(L.oz2o_f32_sub(a, b, up)) == _round_dir(fa - fb, bool(up))
            assert np.float32(L.oz2o_f32_mul(a, b, up)) == _round_dir(fa * fb, bool(up))
            assert np.float32(L.oz2o_f32_fma(a, b, c, up)) == _round_dir(fa * fb + fc, bool(up))


def test_f32_from_u64_round_up():
    L = O.lib()
    rng = random.Random(3)
    vals = [1, 2, 3, (1 << 24) - 1, 1 << 24, (1 << 24) + 1, (1 << 63), (1 << 63) - 1, (1 << 44) * 1024 + 1]
    vals += [rng.randrange(1, 1 << rng.randrange(1, 64)) for _ in range(3000)]
    for v in vals:
        f = np.float32(L.oz2o_f32_from_u64_up(v))
        assert Fraction(float(f)) >= v
        assert Fraction(float(np.nextafter(f, np.float32(0)))) < v


# ------------------------------------------------------------------ integer -> double rounding (R8)
def test_words_to_double_is_correctly_rounded():
    rng = random.Random(11)
    cases = []
    for _ in range(4000):
        bits = rng.randrange(1, 200)
        v = rng.randrange(1 << (bits - 1), 1 << bits)
        if rng.random() < 0.5:
            v = -v
        sh = rng.randrange(-1300, 900)
        cases.append((v, sh))
    # ties and near-ties around 53 bits, subnormal results, overflow
    for t in (54, 55, 60, 100, 160):
        base = (1 << (t - 1)) | (1 << (t - 54))        # exactly half an ulp above a double
        cases += [(base, 0), (base + 1, 0), (base - 1, 0), (-(base | (1 << (t - 53))), 3)]
    cases += [(1, -1074), (1, -1075), (3, -1076), ((1 << 60) + 1, -1130), ((1 << 100) - 1, -1170),
              ((1 << 53) - 1, 971), ((1 << 54) - 1, 970), (1 << 10, 1020)]
    for v, sh in cases:
        got = O.words_to_double(O.int_to_words(v), sh)
        x = Fraction(v) * (Fraction(2) ** sh)
        try:
            want = float(x)                             # CPython: correctly rounded, ties to even
        except OverflowError:
            want = math.inf if v > 0 else -math.inf
        assert got == want, (v, sh, got, want)
