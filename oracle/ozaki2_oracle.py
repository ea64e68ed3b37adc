"""ctypes binding of the CPU oracle (oracle/ozaki2_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this.  It never imports the CUDA package.
Argument marshalling only for the real entry points (every number is computed by the C file); the complex variants
zgemm / cgemm are DEFINED here: numpy embedding, the C oracle on it, and the complex alpha / beta tail in numpy.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

MODE_ACCURATE, MODE_FAST, MODE_PROP = 0, 1, 2
MAX_MODULI = 20


def lib():
    global _LIB
    if _LIB is None:
        from . import build as _build  # compiling the checker is not using it

        _LIB = C.CDLL(_build.build())
        L = _LIB
        L.oz2o_log2f.restype = C.c_float
        L.oz2o_log2f.argtypes = [C.c_float]
        for nm in ("oz2o_f32_add", "oz2o_f32_sub", "oz2o_f32_mul"):
            getattr(L, nm).restype = C.c_float
            getattr(L, nm).argtypes = [C.c_float, C.c_float, C.c_int]
        L.oz2o_f32_fma.restype = C.c_float
        L.oz2o_f32_fma.argtypes = [C.c_float, C.c_float, C.c_float, C.c_int]
        L.oz2o_f32_from_u64_up.restype = C.c_float
        L.oz2o_f32_from_u64_up.argtypes = [C.c_uint64]
        L.oz2o_words_to_double.restype = C.c_double
        L.oz2o_words_to_double.argtypes = [C.c_void_p, C.c_long]
        L.oz2o_num_threads.restype = C.c_int
        L.oz2o_words_to_float.restype = C.c_float
        L.oz2o_words_to_float.argtypes = [C.c_void_p, C.c_long]
    return _LIB


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f(a):
    a = np.asarray(a, dtype=np.float64)
    if not a.flags.f_contiguous:
        a = np.asfortranarray(a)
    return a


def words_to_int(words) -> int:
    """4 little-endian u64 words (two's complement) -> Python int."""
    v = 0
    for t in range(4):
        v |= int(words[t]) << (64 * t)
    if v >> 255:
        v -= 1 << 256
    return v


def words_array_to_ints(arr):
    """[..., 4] uint64 -> object array of Python ints."""
    flat = arr.reshape(-1, 4)
    out = np.empty(flat.shape[0], dtype=object)
    for t in range(flat.shape[0]):
        out[t] = words_to_int(flat[t])
    return out.reshape(arr.shape[:-1])


def pairs_to_ints(arr):
    """[..., 2] uint64 (lo, hi of a two's-complement int128) -> object array of ints."""
    flat = arr.reshape(-1, 2)
    out = np.empty(flat.shape[0], dtype=object)
    for t in range(flat.shape[0]):
        v = int(flat[t, 0]) | (int(flat[t, 1]) << 64)
        if v >> 127:
            v -= 1 << 128
        out[t] = v
    return out.reshape(arr.shape[:-1])


def constants(N: int) -> dict:
    p = np.zeros(MAX_MODULI, np.int32)
    q = np.zeros(MAX_MODULI, np.int32)
    P = np.zeros(4, np.uint64)
    w = np.zeros((MAX_MODULI, 4), np.uint64)
    pp, pf, dl = C.c_float(), C.c_float(), C.c_float()
    rc = lib().oz2o_constants(C.c_int(N), _p(p), _p(q), _p(P), _p(w), C.byref(pp), C.byref(pf), C.byref(dl))
    if rc:
        raise ValueError(f"oz2o_constants({N}) -> {rc}")
    return dict(N=N, p=[int(x) for x in p[:N]], q=[int(x) for x in q[:N]], P=words_to_int(P),
                w=[words_to_int(w[l]) for l in range(N)],
                Pprop=np.float32(pp.value), Pfast=np.float32(pf.value), delta=np.float32(dl.value))


def log2f(x) -> np.float32:
    return np.float32(lib().oz2o_log2f(C.c_float(float(x))))


def log2f_array(x):
    x = np.ascontiguousarray(x, np.float32)
    y = np.empty_like(x)
    lib().oz2o_log2f_array(_p(x), _p(y), C.c_long(x.size))
    return y


def exponents(mode: int, N: int, A, B, extras: bool = False):
    """e[m], f[n] (log2 mu_i, log2 nu_j).  extras=True also returns the statistics."""
    A, B = _f(A), _f(B)
    m, k = A.shape
    k2, n = B.shape
    assert k == k2
    e = np.zeros(m, np.int32)
    f = np.zeros(n, np.int32)
    EA = np.zeros(m, np.int32)
    EB = np.zeros(n, np.int32)
    SA = np.zeros(m, np.uint64)
    SB = np.zeros(n, np.uint64)
    rm = np.zeros(m, np.int64)
    cm = np.zeros(n, np.int64)
    rc = lib().oz2o_exponents(C.c_int(mode), C.c_int(N), C.c_long(m), C.c_long(n), C.c_long(k),
                              _p(A), C.c_long(max(1, m)), _p(B), C.c_long(max(1, k)),
                              _p(e), _p(f), _p(EA), _p(EB), _p(SA), _p(SB), _p(rm), _p(cm))
    if rc:
        raise ValueError(f"oz2o_exponents -> {rc}")
    if extras:
        return e, f, dict(EA=EA, EB=EB, SA=SA, SB=SB, rowmax=rm, colmax=cm)
    return e, f


def truncate(op: int, X, ex):
    """A' (op=0: rows of A -> [m][k]) or B' (op=1: columns of B -> [n][k]) as Python ints."""
    X = _f(X)
    rows, k = (X.shape[0], X.shape[1]) if op == 0 else (X.shape[1], X.shape[0])
    out = np.zeros((rows, k, 2), np.uint64)
    ex = np.ascontiguousarray(ex, np.int32)
    rc = lib().oz2o_truncate(C.c_int(op), C.c_long(rows), C.c_long(k), _p(X), C.c_long(max(1, X.shape[0])),
                             _p(ex), _p(out))
    if rc:
        raise ValueError(f"oz2o_truncate -> {rc}")
    return out


def residues(op: int, N: int, X, ex):
    """INT8 residue planes [N][rows][k] (k fastest)."""
    X = _f(X)
    rows, k = (X.shape[0], X.shape[1]) if op == 0 else (X.shape[1], X.shape[0])
    out = np.zeros((N, rows, k), np.int8)
    ex = np.ascontiguousarray(ex, np.int32)
    rc = lib().oz2o_residues(C.c_int(op), C.c_int(N), C.c_long(rows), C.c_long(k), _p(X),
                             C.c_long(max(1, X.shape[0])), _p(ex), _p(out))
    if rc:
        raise ValueError(f"oz2o_residues -> {rc}")
    return out


def products(N: int, RA, RB):
    """U[N][n][m] uint8 (m fastest) and max |R_l| over everything."""
    RA = np.ascontiguousarray(RA, np.int8)
    RB = np.ascontiguousarray(RB, np.int8)
    _, m, k = RA.shape
    _, n, _ = RB.shape
    U = np.zeros((N, n, m), np.uint8)
    mx = C.c_int64()
    rc = lib().oz2o_products(C.c_int(N), C.c_long(m), C.c_long(n), C.c_long(k), _p(RA), _p(RB), _p(U), C.byref(mx))
    if rc:
        raise ValueError(f"oz2o_products -> {rc}")
    return U, int(mx.value)


def crt(N: int, U):
    """C'' as [n][m][4] uint64 words."""
    U = np.ascontiguousarray(U, np.uint8)
    _, n, m = U.shape
    out = np.zeros((n, m, 4), np.uint64)
    rc = lib().oz2o_crt(C.c_int(N), C.c_long(m), C.c_long(n), _p(U), _p(out))
    if rc:
        raise ValueError(f"oz2o_crt -> {rc}")
    return out


def exact_product(N: int, Ap, Bp, want_words: bool = True):
    """Exact Z = A'B', Zabs = sum|a'||b'| ([n][m][4] words) and the condition-(1) counts."""
    m, k, _ = Ap.shape
    n = Bp.shape[0]
    Z = np.zeros((n, m, 4), np.uint64) if want_words else None
    Za = np.zeros((n, m, 4), np.uint64) if want_words else None
    counts = np.zeros(2, np.int64)
    rc = lib().oz2o_exact_product(C.c_int(N), C.c_long(m), C.c_long(n), C.c_long(k), _p(Ap), _p(Bp),
                                  _p(Z), _p(Za), _p(counts))
    if rc:
        raise ValueError(f"oz2o_exact_product -> {rc}")
    return Z, Za, dict(violations=int(counts[0]), wrong=int(counts[1]))


def unscale(Cpp, e, f, alpha: float = 1.0, beta: float = 0.0, C_in=None):
    n, m, _ = Cpp.shape
    out = np.zeros((m, n), np.float64, order="F") if C_in is None else np.array(C_in, np.float64, order="F")
    e = np.ascontiguousarray(e, np.int32)
    f = np.ascontiguousarray(f, np.int32)
    rc = lib().oz2o_unscale(C.c_long(m), C.c_long(n), _p(Cpp), _p(e), _p(f), C.c_double(alpha), C.c_double(beta),
                            _p(out), C.c_long(max(1, m)))
    if rc:
        raise ValueError(f"oz2o_unscale -> {rc}")
    return out


def unscale_f32(Cpp, e, f, alpha: float = 1.0, beta: float = 0.0, C_in=None):
    """FP32 tail of the SGEMM variant (marshalling of oz2o_unscale_f32): RN_32(C'' 2^-(e_i+f_j)), alpha / beta in FP32."""
    n, m, _ = Cpp.shape
    out = np.zeros((m, n), np.float32, order="F") if C_in is None else np.array(C_in, np.float32, order="F")
    e = np.ascontiguousarray(e, np.int32)
    f = np.ascontiguousarray(f, np.int32)
    rc = lib().oz2o_unscale_f32(C.c_long(m), C.c_long(n), _p(Cpp), _p(e), _p(f), C.c_float(alpha), C.c_float(beta),
                                _p(out), C.c_long(max(1, m)))
    if rc:
        raise ValueError(f"oz2o_unscale_f32 -> {rc}")
    return out


def words_to_double(words, sh: int) -> float:
    words = np.ascontiguousarray(words, np.uint64)
    return float(lib().oz2o_words_to_double(_p(words), C.c_long(sh)))


def int_to_words(v: int):
    v &= (1 << 256) - 1
    return np.array([(v >> (64 * t)) & 0xFFFFFFFFFFFFFFFF for t in range(4)], np.uint64)


def dgemm(A, B, N: int, mode: int, alpha: float = 1.0, beta: float = 0.0, C_in=None, return_exponents=False):
    """The whole path (Steps 1-4) in one call."""
    A, B = _f(A), _f(B)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float64, order="F") if C_in is None else np.array(C_in, np.float64, order="F")
    e = np.zeros(max(1, m), np.int32)
    f = np.zeros(max(1, n), np.int32)
    rc = lib().oz2o_dgemm(C.c_long(m), C.c_long(n), C.c_long(k), C.c_double(alpha), _p(A), C.c_long(max(1, m)),
                          _p(B), C.c_long(max(1, k)), C.c_double(beta), _p(out), C.c_long(max(1, m)),
                          C.c_int(N), C.c_int(mode), _p(e), _p(f))
    if rc:
        raise ValueError(f"oz2o_dgemm -> {rc}")
    if return_exponents:
        return out, e[:m], f[:n]
    return out


def words_to_float(words, sh: int) -> np.float32:
    words = np.ascontiguousarray(words, np.uint64)
    return np.float32(lib().oz2o_words_to_float(_p(words), C.c_long(sh)))


def sgemm(A, B, N: int, mode: int, alpha: float = 1.0, beta: float = 0.0, C_in=None, return_exponents=False):
    """SGEMM variant (Fig. 6): FP32 in / FP32 out, Steps 1-3 on the promoted inputs, one rounding to FP32."""
    A = np.asfortranarray(np.asarray(A, dtype=np.float32))
    B = np.asfortranarray(np.asarray(B, dtype=np.float32))
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float32, order="F") if C_in is None else np.array(C_in, np.float32, order="F")
    e = np.zeros(max(1, m), np.int32)
    f = np.zeros(max(1, n), np.int32)
    rc = lib().oz2o_sgemm(C.c_long(m), C.c_long(n), C.c_long(k), C.c_float(alpha), _p(A), C.c_long(max(1, m)),
                          _p(B), C.c_long(max(1, k)), C.c_float(beta), _p(out), C.c_long(max(1, m)),
                          C.c_int(N), C.c_int(mode), _p(e), _p(f))
    if rc:
        raise ValueError(f"oz2o_sgemm -> {rc}")
    if return_exponents:
        return out, e[:m], f[:n]
    return out


def zgemm_embedding(A, B):
    """Real embedding of a complex product (DESIGN.md 8b #4): [C_r; C_i] = [[A_r, -A_i], [A_i, A_r]] [B_r; B_i]."""
    A = np.asarray(A, dtype=np.complex128)
    B = np.asarray(B, dtype=np.complex128)
    At = np.block([[A.real, -A.imag], [A.imag, A.real]])
    Bt = np.vstack([B.real, B.imag])
    return np.asfortranarray(At), np.asfortranarray(Bt)


def zgemm(A, B, N: int, mode: int, alpha: complex = 1.0, beta: complex = 0.0, C_in=None):
    """Complex variant (named as future work at P:58; reading in DESIGN.md 8b #4): oz2o_dgemm on the real embedding,
    then out = alpha c + beta C_in in plain complex arithmetic -- every product and every sum rounded on its own, in the
    order written below; alpha == 1, beta == 0 and beta == 1 are not multiplied (BLAS rules: beta == 0 overwrites, beta == 1
    adds C_in as it is -- for finite C_in the same bits as 1 * C_in, but an Inf or NaN in one part of an entry no longer
    reaches the other part through 0 * Inf)."""
    A = np.asarray(A, dtype=np.complex128)
    B = np.asarray(B, dtype=np.complex128)
    m = A.shape[0]
    At, Bt = zgemm_embedding(A, B)
    Ct = dgemm(At, Bt, N, mode)
    cr, ci = Ct[:m], Ct[m:]
    alpha, beta = complex(alpha), complex(beta)
    if alpha != 1.0:
        with np.errstate(all="ignore"):
            tr = alpha.real * cr - alpha.imag * ci
            ti = alpha.real * ci + alpha.imag * cr
    else:
        tr, ti = cr, ci
    if beta == 1.0:
        Cin = np.asarray(C_in, dtype=np.complex128)
        with np.errstate(all="ignore"):
            tr, ti = tr + Cin.real, ti + Cin.imag
    elif beta != 0.0:
        Cin = np.asarray(C_in, dtype=np.complex128)
        with np.errstate(all="ignore"):
            tr = tr + (beta.real * Cin.real - beta.imag * Cin.imag)
            ti = ti + (beta.real * Cin.imag + beta.imag * Cin.real)
    out = np.empty(cr.shape, np.complex128, order="F")
    out.real, out.imag = tr, ti
    return out


def cgemm(A, B, N: int, mode: int, alpha: complex = 1.0, beta: complex = 0.0, C_in=None):
    """Single-precision complex variant (same reading as zgemm, DESIGN.md 8b #4): oz2o_sgemm on the real embedding of the FP32
    parts, then out = alpha c + beta C_in in FP32 complex arithmetic -- every product and every sum rounded to FP32 on its own,
    in the order written below; alpha == 1, beta == 0 and beta == 1 are not multiplied."""
    A = np.asarray(A, dtype=np.complex64)
    B = np.asarray(B, dtype=np.complex64)
    m = A.shape[0]
    At = np.asfortranarray(np.block([[A.real, -A.imag], [A.imag, A.real]]).astype(np.float32))
    Bt = np.asfortranarray(np.vstack([B.real, B.imag]).astype(np.float32))
    Ct = sgemm(At, Bt, N, mode)
    cr, ci = Ct[:m], Ct[m:]
    alpha, beta = complex(alpha), complex(beta)
    f = np.float32
    if alpha != 1.0:
        ar, ai = f(alpha.real), f(alpha.imag)
        with np.errstate(all="ignore"):
            tr = (ar * cr).astype(f) - (ai * ci).astype(f)
            ti = (ar * ci).astype(f) + (ai * cr).astype(f)
    else:
        tr, ti = cr, ci
    if beta == 1.0:
        Cin = np.asarray(C_in, dtype=np.complex64)
        with np.errstate(all="ignore"):
            tr, ti = tr + Cin.real, ti + Cin.imag
    elif beta != 0.0:
        Cin = np.asarray(C_in, dtype=np.complex64)
        br, bi = f(beta.real), f(beta.imag)
        with np.errstate(all="ignore"):
            tr = tr + ((br * Cin.real).astype(f) - (bi * Cin.imag).astype(f))
            ti = ti + ((br * Cin.imag).astype(f) + (bi * Cin.real).astype(f))
    out = np.empty(cr.shape, np.complex64, order="F")
    out.real, out.imag = tr, ti
    return out


def dd_reference(A, B):
    """AB in double-double: (hi, lo), each (m, n) column-major."""
    A, B = _f(A), _f(B)
    m, k = A.shape
    _, n = B.shape
    hi = np.zeros((m, n), np.float64, order="F")
    lo = np.zeros((m, n), np.float64, order="F")
    lib().oz2o_dd_reference(C.c_long(m), C.c_long(n), C.c_long(k), _p(A), C.c_long(max(1, m)), _p(B),
                            C.c_long(max(1, k)), _p(hi), _p(lo))
    return hi, lo


def num_threads() -> int:
    return int(lib().oz2o_num_threads())


def stages(A, B, N: int, mode: int, want_exact: bool = False) -> dict:
    """Every stage of the path on (A, B): exponents, residues, products, C'', C."""
    A, B = _f(A), _f(B)
    e, f, ext = exponents(mode, N, A, B, extras=True)
    RA = residues(0, N, A, e)
    RB = residues(1, N, B, f)
    U, maxR = products(N, RA, RB)
    Cpp = crt(N, U)
    Cout = unscale(Cpp, e, f)
    out = dict(e=e, f=f, RA=RA, RB=RB, U=U, maxR=maxR, Cpp=Cpp, C=Cout, **ext)
    if want_exact:
        Ap = truncate(0, A, e)
        Bp = truncate(1, B, f)
        Z, Za, cnt = exact_product(N, Ap, Bp)
        out.update(Ap=Ap, Bp=Bp, Z=Z, Zabs=Za, counts=cnt)
    return out
