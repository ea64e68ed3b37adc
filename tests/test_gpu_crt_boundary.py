"""GPU parity of S4 + S5 on CHOSEN residues (-m gpu): ozaki2_debug_crt feeds caller-made U planes into the CRT
kernel of ozaki2_dgemm, so that the boundary cases of eq. (3) (reading R7: C'' in [-P/2, P/2)) reach the
hardware: values at and around +-P/2, quotient estimates within 2^-20 of a half-integer (the hand-over from the
branch-free common case to the exact routine), small and zero values, and exponents that make the result normal,
subnormal and overflowing -- for every moduli count (all five word counts of P), FP64 and FP32 outputs, with and
without the C'' output (exact routine for every element / production code path).  Expected values come from the
oracle (crt, unscale) and from Python integers."""
import random

import numpy as np
import pytest

from oracle import ozaki2_oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_29129_b200 as pkg
    pkg.lib()
    return pkg


def boundary_integers(N, count_random, seed):
    P = O.constants(N)["P"]
    h = P // 2
    step = max(1, P >> 21)
    zs = [0, 1, -1, 2, -2, h - 1, -h, h, -h - 1, h - 2, -h + 1, 3 * P + 7, -3 * P - 7, P, -P, P - 1, 255 * 20 * P // 3]
    for t in range(5):
        for sgn in (1, -1):
            for d in (t * step, -t * step, t, -t):
                zs.append(sgn * h + d)
    # every magnitude class (leading bit 0 .. log2 P - 2: all word positions of the normalisation) and the rounding
    # patterns of RN_64 / RN_32 at each of them: exact ties (round to even both ways), ties broken by a sticky bit far
    # below, all-ones carries into the next binade
    L = P.bit_length() - 2
    for bpos in range(0, L + 1):
        for v in ((1 << bpos), (1 << bpos) - 1, (1 << bpos) + 1):
            if 0 < v < h:
                zs.extend((v, -v))
    for prec in (53, 24):
        for sh in list(range(1, max(2, L - prec), 5)) + [max(1, L - prec - 1)]:
            for mant in ((1 << prec) | 1, (1 << prec) | 3, (1 << (prec + 1)) - 1, (1 << prec) + 2):
                base = (mant << sh) >> 1                      # prec + 1 significant bits: the last one is the round bit
                for v in (base, base + 1, base - 1, base + (1 << (sh // 2)), base - (1 << (sh // 2))):
                    if 0 < v < h:
                        zs.extend((v, -v))
    rng = random.Random(seed)
    win = max(2, P >> 20)
    for _ in range(count_random):                     # within P 2^-20 of +-P/2: the near-half quotient window
        zs.append(rng.choice((1, -1)) * h + rng.randrange(-win, win))
    for _ in range(count_random // 4):                # ordinary values, small values, a few multiples of P away
        zs.append(rng.randrange(-h, h))
        zs.append(rng.randrange(-(1 << 20), 1 << 20))
        zs.append(rng.randrange(-h, h) + rng.randrange(-4000, 4000) * P)
    return zs, P


def planes_from_integers(N, zs, m, n):
    p = O.constants(N)["p"]
    z = np.array(zs, dtype=object)
    U = np.zeros((N, n * m), np.uint8)
    for l, q in enumerate(p):
        U[l, :len(zs)] = np.array([int(v % q) for v in zs], np.uint8)
    return U.reshape(N, n, m)


@pytest.mark.parametrize("N", range(2, 21))
def test_crt_kernel_on_boundary_residues(B, N):
    import torch
    m, n = 272, 96                                    # 26112 elements, m = 16 * 17: ragged against the 512-row tile
    zs, P = boundary_integers(N, 10000, 100 + N)
    assert len(zs) <= m * n
    U = planes_from_integers(N, zs, m, n)
    want_int = [((int(v) + P // 2) % P) - P // 2 for v in zs]
    Cpp_o = O.crt(N, U)                                                         # [n][m][4]
    flat = Cpp_o.reshape(-1, 4)
    for t in (0, 1, 5, 7, 8, 11, len(zs) - 1):                                   # the oracle itself against Python integers
        assert O.words_to_int(flat[t]) == want_int[t]
    Ud = torch.from_numpy(U).cuda()
    rng = np.random.Generator(np.random.PCG64(N))
    lgP = P.bit_length()
    cases = [("normal", rng.integers(-40, 40, size=m), rng.integers(-40, 40, size=n)),
             ("subnormal", rng.integers(1040, 1075, size=m) + lgP // 2, rng.integers(0, 10, size=n) + lgP // 2),
             ("overflow", -rng.integers(985, 1000, size=m), -rng.integers(0, 40, size=n))]
    for tag, e, f in cases:
        e, f = e.astype(np.int32), f.astype(np.int32)
        ed, fd = torch.from_numpy(e).cuda(), torch.from_numpy(f).cuda()
        for f32 in (False, True):
            if f32:
                e2, f2 = (e // 8).astype(np.int32), (f // 8).astype(np.int32)     # FP32 range: the same three regimes
                ed, fd = torch.from_numpy(e2).cuda(), torch.from_numpy(f2).cuda()
                want = O.unscale_f32(Cpp_o, e2, f2)
                dt = torch.float32
            else:
                want = O.unscale(Cpp_o, e, f)
                dt = torch.float64
            for with_cpp in (True, False):
                Cd = torch.full((n, m), float("nan"), dtype=dt, device="cuda")
                Cppd = torch.zeros((n, m, 4), dtype=torch.int64, device="cuda") if with_cpp else None
                rc = B.ozaki2_debug_crt(N, m, n, Ud, ed, fd, 1.0, 0.0, Cd, m, Cppd, f32)
                assert rc == 0
                torch.cuda.synchronize()
                got = B.device_to_colmajor(Cd)
                with np.errstate(all="ignore"):
                    assert np.array_equal(got, want), (N, tag, f32, with_cpp, int(np.sum(got != want)))
                if with_cpp:
                    assert np.array_equal(Cppd.cpu().numpy().view(np.uint64), Cpp_o), (N, tag, f32)


def test_crt_kernel_alpha_beta_and_arguments(B):
    import torch
    N, m, n = 14, 32, 5
    zs, P = boundary_integers(N, 100, 3)
    zs = zs[:m * n]
    U = planes_from_integers(N, zs, m, n)
    Cpp_o = O.crt(N, U)
    e = np.arange(m, dtype=np.int32) - 10
    f = np.arange(n, dtype=np.int32) + 50
    rng = np.random.Generator(np.random.PCG64(8))
    ldc = m + 8
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)))
    Ud, ed, fd = torch.from_numpy(U).cuda(), torch.from_numpy(e).cuda(), torch.from_numpy(f).cuda()
    Cd = B.colmajor_to_device(Cin)
    assert B.ozaki2_debug_crt(N, m, n, Ud, ed, fd, -0.75, 2.5, Cd, ldc) == 0
    torch.cuda.synchronize()
    got = B.device_to_colmajor(Cd)
    assert np.array_equal(got[:m], O.unscale(Cpp_o, e, f, alpha=-0.75, beta=2.5, C_in=Cin[:m].copy()))
    assert np.array_equal(got[m:], Cin[m:])
    assert B.ozaki2_debug_crt(1, m, n, Ud, ed, fd, 1.0, 0.0, Cd, ldc) == -1
    assert B.ozaki2_debug_crt(N, m + 1, n, Ud, ed, fd, 1.0, 0.0, Cd, ldc) == -2
    assert B.ozaki2_debug_crt(N, m, n, Ud, ed, fd, 1.0, 0.0, Cd, m - 1) == -10


def test_crt_kernel_more_row_blocks_than_resident_ctas(B):
    """m beyond (resident CTAs) x 512 rows: the launcher covers the row blocks in several launches."""
    import torch
    N, m, n = 5, 148 * 3 * 512 + 704, 3              # m % 16 == 0: the debug entry uses the planes in place
    rng = np.random.Generator(np.random.PCG64(77))
    U = np.stack([rng.integers(0, q, size=(n, m), dtype=np.int64).astype(np.uint8) for q in O.constants(N)["p"]])
    Cpp_o = O.crt(N, U)
    e = rng.integers(-30, 30, size=m).astype(np.int32)
    f = rng.integers(-30, 30, size=n).astype(np.int32)
    want = O.unscale(Cpp_o, e, f)
    Ud, ed, fd = torch.from_numpy(U).cuda(), torch.from_numpy(e).cuda(), torch.from_numpy(f).cuda()
    Cd = torch.full((n, m), float("nan"), dtype=torch.float64, device="cuda")
    assert B.ozaki2_debug_crt(N, m, n, Ud, ed, fd, 1.0, 0.0, Cd, m) == 0
    torch.cuda.synchronize()
    assert np.array_equal(B.device_to_colmajor(Cd), want)
