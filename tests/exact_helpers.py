"""Exact-rational helpers for the pin tests (no oracle, no CUDA code in here)."""
import math
from fractions import Fraction

import numpy as np


def floor_log2(v: float) -> int:
    _, e = math.frexp(abs(v))
    return e - 1


def frac_sumsq(vec) -> Fraction:
    return sum(Fraction(float(x)) ** 2 for x in vec)


def pow2(e: int) -> Fraction:
    return Fraction(2) ** int(e)


def round_dir_f32(x: Fraction, up: bool) -> np.float32:
    """Exact rational -> float32 rounded toward +inf (up) or -inf (down)."""
    if x == 0:
        return np.float32(0.0)
    f = np.float32(float(x))
    while Fraction(float(f)) < x:
        f = np.nextafter(f, np.float32(np.inf))
    while Fraction(float(f)) > x:
        f = np.nextafter(f, np.float32(-np.inf))
    if up and Fraction(float(f)) < x:
        f = np.nextafter(f, np.float32(np.inf))
    return np.float32(f)


def trunc_scaled(a: float, e: int) -> int:
    """trunc(a * 2^e) in exact rational arithmetic (Step 2)."""
    return math.trunc(Fraction(float(a)) * pow2(e))


def sym_mod(v: int, p: int) -> int:
    """Symmetric residue: v mod p mapped to [-(p-1)//2 .. p//2] with p = 256 -> [-128, 127]."""
    u = v % p
    return u - p if u > (p - 1) // 2 else u
