"""GPU parity of the remaining entry points (-m gpu): the plain ozaki2_dgemm / ozaki2_sgemm calls (production CRT code
path, no stage outputs) on inputs whose results are subnormal, overflowing or spread over the whole exponent range;
the full BLAS shape (row-major, 'N' / 'T' / 'C'); ozaki2_sgemm_t; ozaki2_sgemm_host.  Expected values: the oracle on
the LOGICAL matrices."""
import numpy as np
import pytest

import workloads as W
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


def plain_dgemm(B, A, Bm, N, mode):
    import torch
    Ad, Bd = B.colmajor_to_device(A), B.colmajor_to_device(Bm)
    Cd = B.dgemm(Ad, Bd, N, mode)
    torch.cuda.synchronize()
    return B.device_to_colmajor(Cd)


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("N", [8, 14, 17, 20])
def test_plain_call_on_wide_exponent_inputs(B, mode, N):
    A, Bm = W.wide_exponent_matrices(300, 130, 260, seed=31 + N)
    with np.errstate(all="ignore"):
        assert np.array_equal(plain_dgemm(B, A, Bm, N, mode), O.dgemm(A, Bm, N, mode))


@pytest.mark.parametrize("sa,sb", [(-600, -500), (600, 500), (-530, -520), (-1000, -40), (500, 523)])
@pytest.mark.parametrize("N", [12, 16, 19])
def test_plain_call_with_subnormal_and_overflowing_results(B, sa, sb, N):
    # C = A B 2^(sa+sb): subnormal, partly flushed to zero, or overflowing; the production CRT path must hand these
    # elements to its exact routine (one rounding in total, also when the result is subnormal)
    A, Bm = W.eq15_matrices(260, 70, 200, 1.0, 900 + N)
    A, Bm = np.ldexp(A, sa), np.ldexp(Bm, sb)
    with np.errstate(all="ignore"):
        want = O.dgemm(A, Bm, N, 2)
        got = plain_dgemm(B, A, Bm, N, 2)
        assert np.array_equal(got, want)
    if -1074 < sa + sb < -1000:
        assert np.any((want != 0) & (np.abs(want) < 2.3e-308))          # subnormal results are really exercised
    if sa + sb > 1000:
        assert np.any(np.isinf(want))


@pytest.mark.parametrize("sa,sb", [(-80, -60), (70, 55)])
def test_plain_sgemm_with_subnormal_and_overflowing_results(B, sa, sb):
    import torch
    A, Bm = W.eq15_matrices(260, 70, 200, 1.0, 77)
    A = np.asfortranarray(np.ldexp(A, sa).astype(np.float32))
    Bm = np.asfortranarray(np.ldexp(Bm, sb).astype(np.float32))
    m, k = A.shape
    n = Bm.shape[1]
    Ad, Bd = B.colmajor_to_device(A, np.float32), B.colmajor_to_device(Bm, np.float32)
    Cd = torch.empty((n, m), dtype=torch.float32, device="cuda")
    B.ensure_workspace(m, n, k, 8, 2)
    assert B.ozaki2_sgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, 8, 2) == 0
    torch.cuda.synchronize()
    with np.errstate(all="ignore"):
        want = O.sgemm(A, Bm, 8, 2)
        assert np.array_equal(B.device_to_colmajor(Cd), want)
    assert np.any(np.isinf(want)) or np.any((want != 0) & (np.abs(want) < 1.2e-38))


def _stored(X, trans, row_major, pad):
    """memory image of logical matrix X under (trans, layout) as a numpy array whose C-order bytes are the buffer,
    and its leading dimension"""
    S = X.T if trans else X                        # the stored matrix
    if row_major:
        ld = S.shape[1] + pad
        buf = np.zeros((S.shape[0], ld), X.dtype)
        buf[:, :S.shape[1]] = S
    else:
        ld = S.shape[0] + pad
        buf = np.zeros((S.shape[1], ld), X.dtype)   # column-major: columns are contiguous
        buf[:, :S.shape[0]] = S.T
    return buf, ld


@pytest.mark.parametrize("layout", ["C", "R", 101])
@pytest.mark.parametrize("ta,tb", [("N", "N"), ("T", "n"), ("n", "C"), ("t", "T"), (111, 112)])
@pytest.mark.parametrize("f32", [False, True])
def test_full_blas_signature(B, layout, ta, tb, f32):
    import torch
    m, n, k, N, mode = 150, 90, 260, (8 if f32 else 15), 2
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 321)
    dt = np.float32 if f32 else np.float64
    A, Bm = np.asfortranarray(A.astype(dt)), np.asfortranarray(Bm.astype(dt))
    rm = layout in ("R", "r", 101)
    tra = ta in ("T", "t", "C", "c", 112, 113)
    trb = tb in ("T", "t", "C", "c", 112, 113)
    bufA, lda = _stored(A, tra, rm, 3)
    bufB, ldb = _stored(Bm, trb, rm, 5)
    rng = np.random.Generator(np.random.PCG64(1))
    Cin = rng.standard_normal((m, n)).astype(dt)
    bufC, ldc = _stored(Cin, False, rm, 2)
    Ad, Bd, Cd = torch.from_numpy(bufA).cuda(), torch.from_numpy(bufB).cuda(), torch.from_numpy(bufC.copy()).cuda()
    B.ensure_workspace(max(m, n), max(m, n), k, N, mode)
    call = B.ozaki2_sgemm_blas if f32 else B.ozaki2_dgemm_blas
    alpha, beta = 0.5, -2.0
    assert call(layout, ta, tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == 0
    torch.cuda.synchronize()
    got = Cd.cpu().numpy()
    got = got[:, :n] if rm else got[:, :m].T
    want = (O.sgemm if f32 else O.dgemm)(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin.copy())
    assert np.array_equal(got, want)
    # errors are reported in the numbering of this prototype, for the caller's own A and B
    assert call("X", ta, tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == -1
    assert call(layout, "Q", tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == -2
    assert call(layout, ta, 7, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == -3
    assert call(layout, ta, tb, -1, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == -4
    assert call(layout, ta, tb, m, -1, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == -5
    assert call(layout, ta, tb, m, n, k, alpha, Ad, 1, Bd, ldb, beta, Cd, ldc, N, mode) == -9
    assert call(layout, ta, tb, m, n, k, alpha, Ad, lda, Bd, 1, beta, Cd, ldc, N, mode) == -11
    assert call(layout, ta, tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, 1, N, mode) == -14
    assert call(layout, ta, tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, 1, mode) == -15
    assert call(layout, ta, tb, m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, 9) == -16


@pytest.mark.parametrize("transa,transb", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_sgemm_transposed_operands(B, transa, transb):
    import torch
    m, n, k, N, mode = 130, 70, 200, 9, 0
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 11)
    A, Bm = np.asfortranarray(A.astype(np.float32)), np.asfortranarray(Bm.astype(np.float32))
    bufA, lda = _stored(A, transa, False, 1)
    bufB, ldb = _stored(Bm, transb, False, 4)
    Ad, Bd = torch.from_numpy(bufA).cuda(), torch.from_numpy(bufB).cuda()
    Cd = torch.full((n, m), float("nan"), dtype=torch.float32, device="cuda")
    B.ensure_workspace(m, n, k, N, mode)
    assert B.ozaki2_sgemm_t(transa, transb, m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, m, N, mode) == 0
    torch.cuda.synchronize()
    assert np.array_equal(B.device_to_colmajor(Cd), O.sgemm(A, Bm, N, mode))
    assert B.ozaki2_sgemm_t(3, 0, m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, m, N, mode) == -1


@pytest.mark.parametrize("n,mode", [(80, 2), (1100, 2), (1100, 1), (600, 0)])
def test_sgemm_host_buffer_entry_point(B, n, mode):
    # n >= 512 in modes 1, 2: column panels with the copies overlapped; otherwise the plain route
    import torch
    m, k, N = 200, 300, 9
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 55)
    lda, ldb, ldc = m + 4, k + 2, m + 6
    Ah = np.zeros((lda, k), np.float32, order="F"); Ah[:m] = A
    Bh = np.zeros((ldb, n), np.float32, order="F"); Bh[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(4))
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)).astype(np.float32))
    Ch = Cin.copy(order="F")
    B.ensure_workspace(m, n, k, N, mode)
    nbytes = B.ozaki2_host_scratch_bytes(m, n, k)
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    assert B.ozaki2_sgemm_host(m, n, k, 0.5, Ah, lda, Bh, ldb, 1.5, Ch, ldc, N, mode, scratch, nbytes) == 0
    want = O.sgemm(Ah[:m], Bh[:k], N, mode, alpha=0.5, beta=1.5, C_in=Cin[:m].copy())
    assert np.array_equal(Ch[:m], want)
    assert np.array_equal(Ch[m:], Cin[m:])
    assert B.ozaki2_sgemm_host(m, n, k, 0.5, Ah, lda, Bh, ldb, 1.5, Ch, ldc, N, mode, scratch, 16) == -14
    assert "14" in B.ozaki2_status_string(-14)


def _complex_inputs(m, n, k, phi, seed):
    Ar, Br = W.eq15_matrices(m, n, k, phi, seed)
    Ai, Bi = W.eq15_matrices(m, n, k, phi, seed + 1)
    return np.asfortranarray(Ar + 1j * Ai), np.asfortranarray(Br + 1j * Bi)


@pytest.mark.parametrize("m,n,k,N,mode,alpha,beta", [
    (70, 50, 90, 14, 2, 1.0, 0.0), (129, 33, 257, 17, 2, 0.5 - 2.0j, -1.25 + 0.75j), (64, 64, 64, 10, 1, 1.0, 1.0),
    (40, 130, 300, 16, 0, -1.0j, 0.0), (1, 1, 1, 2, 2, 1.0, 0.0), (200, 20, 1000, 20, 2, 2.0, 0.5j),
])
def test_zgemm_against_the_oracle_on_the_real_embedding(B, m, n, k, N, mode, alpha, beta):
    # SURVEY 8(f) #4 (reading DESIGN.md 8b #4): bit-exact against oz2o_dgemm on the embedding + the stated tail
    import torch
    A, Bm = _complex_inputs(m, n, k, 1.0, 700 + m + n + k)
    lda, ldb, ldc = m + 3, k + 1, m + 2
    Ap = np.zeros((lda, k), np.complex128, order="F"); Ap[:m] = A
    Bp = np.zeros((ldb, n), np.complex128, order="F"); Bp[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(9))
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)) + 1j * rng.standard_normal((ldc, n)))
    Ad = torch.from_numpy(np.ascontiguousarray(Ap.T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bp.T)).cuda()
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, mode)
    assert B.ozaki2_zgemm(m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == 0
    torch.cuda.synchronize()
    got = np.asfortranarray(Cd.cpu().numpy().T)
    want = O.zgemm(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin[:m])
    assert np.array_equal(got[:m], want)
    assert np.array_equal(got[m:], Cin[m:])
    if mode != 1:
        ref = A @ Bm
        assert np.max(np.abs(O.zgemm(A, Bm, N, mode) - ref) / np.abs(ref)) < {10: 1e-2, 14: 1e-6, 16: 1e-8, 17: 1e-9, 20: 1e-13}.get(N, 1.0)


@pytest.mark.parametrize("cplx,m,n,k,N,mode,alpha,beta", [
    # several ragged waves of every persistent kernel on the embedded (2m x 2k)(2k x n) problem, complex alpha / beta
    ("z", 1100, 700, 1500, 16, 2, 0.5 - 2.0j, -1.25 + 0.75j), ("z", 600, 520, 900, 16, 1, 1.0, 1.0), ("z", 600, 520, 900, 18, 0, -1.0j, 0.0),
    ("c", 1100, 700, 1500, 9, 2, 0.5 - 2.0j, -1.25 + 0.75j), ("c", 600, 520, 900, 9, 1, 1.0, 1.0), ("c", 600, 520, 900, 10, 0, -1.0j, 0.0),
    # n or k beyond 65535 (the grid.y limit the embed / combine kernels once had); 2k > 2^17 also takes the K-blocked GEMM
    ("z", 3, 70000, 5, 8, 2, 1.0, 0.5j), ("z", 2, 3, 66000, 14, 2, 2.0, 0.0), ("c", 2, 66000, 3, 6, 1, 1.0j, 1.0), ("c", 3, 2, 65600, 8, 2, 1.0, 0.0),
])
def test_complex_entries_at_multi_wave_and_long_sizes(B, cplx, m, n, k, N, mode, alpha, beta):
    # bit-exact against the oracle's definition, element by element
    import torch
    ct = np.complex128 if cplx == "z" else np.complex64
    A, Bm = _complex_inputs(m, n, k, 1.0, 1700 + m + n + k)
    A, Bm = np.asfortranarray(A.astype(ct)), np.asfortranarray(Bm.astype(ct))
    lda, ldb, ldc = m + 5, k + 3, m + 1
    Ap = np.zeros((lda, k), ct, order="F"); Ap[:m] = A
    Bp = np.zeros((ldb, n), ct, order="F"); Bp[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(29))
    Cin = np.asfortranarray((rng.standard_normal((ldc, n)) + 1j * rng.standard_normal((ldc, n))).astype(ct))
    Ad = torch.from_numpy(np.ascontiguousarray(Ap.T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bp.T)).cuda()
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, mode)
    call, oracle = (B.ozaki2_zgemm, O.zgemm) if cplx == "z" else (B.ozaki2_cgemm, O.cgemm)
    assert call(m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == 0
    torch.cuda.synchronize()
    got = np.asfortranarray(Cd.cpu().numpy().T)
    want = oracle(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin[:m])
    assert got.dtype == ct and np.array_equal(got[:m], want)
    assert np.array_equal(got[m:], Cin[m:])


@pytest.mark.parametrize("cplx", ["z", "c"])
def test_complex_beta_one_adds_c_as_it_is_and_the_quick_return_leaves_it_alone(B, cplx):
    import torch
    ct, N = (np.complex128, 14) if cplx == "z" else (np.complex64, 8)
    call, oracle = (B.ozaki2_zgemm, O.zgemm) if cplx == "z" else (B.ozaki2_cgemm, O.cgemm)
    m, n, k = 40, 24, 70
    A, Bm = _complex_inputs(m, n, k, 0.5, 77)
    A, Bm = np.asfortranarray(A.astype(ct)), np.asfortranarray(Bm.astype(ct))
    rng = np.random.Generator(np.random.PCG64(5))
    Cin = np.asfortranarray((rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))).astype(ct))
    Cin[3, 4] = complex(np.inf, 2.0)                  # a non-finite part must stay in its own part
    Cin[5, 6] = complex(-1.0, np.nan)
    Cin[7, 8] = complex(-np.inf, -0.0)
    Ad = torch.from_numpy(np.ascontiguousarray(A.T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bm.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, 2)
    word = np.uint64 if cplx == "z" else np.uint32
    for alpha, kk in ((0.0, k), (1.0, 0)):            # quick returns with beta == 1: C is not touched at all
        Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
        before = B.ozaki2_kernel_launches()
        assert call(m, n, kk, alpha, Ad, m, Bd, max(1, kk), 1.0, Cd, m, N, 2) == 0
        torch.cuda.synchronize()
        assert B.ozaki2_kernel_launches() == before
        assert np.array_equal(Cd.cpu().numpy().view(word), np.ascontiguousarray(Cin.T).view(word))
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    assert call(m, n, k, 0.5 - 2.0j, Ad, m, Bd, k, 1.0, Cd, m, N, 2) == 0
    torch.cuda.synchronize()
    got = np.asfortranarray(Cd.cpu().numpy().T)
    want = oracle(A, Bm, N, 2, alpha=0.5 - 2.0j, beta=1.0, C_in=Cin)
    # (NaN payloads are not part of the contract: FP32 adds on the GPU return the canonical NaN)
    assert np.array_equal(got.real, want.real, equal_nan=True) and np.array_equal(got.imag, want.imag, equal_nan=True)
    assert np.isfinite(got[3, 4].imag) and np.isfinite(got[5, 6].real) and got[7, 8].real == -np.inf and np.isfinite(got[7, 8].imag)


def test_zgemm_quick_returns_and_errors(B):
    import torch
    m, n, k, N = 32, 16, 24, 12
    A, Bm = _complex_inputs(m, n, k, 0.5, 3)
    Ad = torch.from_numpy(np.ascontiguousarray(A.T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bm.T)).cuda()
    Cin = np.asfortranarray(np.arange(m * n).reshape(m, n) * (1.0 + 0.5j))
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, 2)
    assert B.ozaki2_zgemm(m, n, k, 0.0, Ad, m, Bd, k, 2.0j, Cd, m, N, 2) == 0        # alpha == 0: C := beta C
    torch.cuda.synchronize()
    assert np.array_equal(np.asfortranarray(Cd.cpu().numpy().T), 2.0j * Cin)
    assert B.ozaki2_zgemm(m, n, 0, 1.0, Ad, m, Bd, 1, 0.0, Cd, m, N, 2) == 0          # k == 0, beta == 0: zeros
    torch.cuda.synchronize()
    assert not np.any(Cd.cpu().numpy())
    assert B.ozaki2_zgemm(-1, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == -1
    assert B.ozaki2_zgemm(m, n, k, 1.0, Ad, m - 1, Bd, k, 0.0, Cd, m, N, 2) == -7
    assert B.ozaki2_zgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, 21, 2) == -14
    assert B.ozaki2_set_workspace(None, 0) == 0
    assert B.ozaki2_zgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == B.OZAKI2_ERR_WORKSPACE


@pytest.mark.parametrize("m,n,k,N,mode,alpha,beta", [
    (70, 50, 90, 8, 2, 1.0, 0.0), (129, 33, 257, 12, 2, 0.5 - 2.0j, -1.25 + 0.75j), (64, 64, 64, 6, 1, 1.0, 1.0),
    (40, 130, 300, 10, 0, -1.0j, 0.0), (1, 1, 1, 2, 2, 1.0, 0.0), (200, 20, 1000, 9, 2, 2.0, 0.5j),
])
def test_cgemm_against_the_oracle_on_the_real_embedding(B, m, n, k, N, mode, alpha, beta):
    # the single-precision complex variant: bit-exact against oz2o_sgemm on the embedding of the FP32 parts + the FP32 tail
    import torch
    A, Bm = _complex_inputs(m, n, k, 1.0, 900 + m + n + k)
    A, Bm = np.asfortranarray(A.astype(np.complex64)), np.asfortranarray(Bm.astype(np.complex64))
    lda, ldb, ldc = m + 3, k + 1, m + 2
    Ap = np.zeros((lda, k), np.complex64, order="F"); Ap[:m] = A
    Bp = np.zeros((ldb, n), np.complex64, order="F"); Bp[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(19))
    Cin = np.asfortranarray((rng.standard_normal((ldc, n)) + 1j * rng.standard_normal((ldc, n))).astype(np.complex64))
    Ad = torch.from_numpy(np.ascontiguousarray(Ap.T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bp.T)).cuda()
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, mode)
    assert B.ozaki2_cgemm_workspace_bytes(m, n, k, N, mode) <= B.ozaki2_zgemm_workspace_bytes(m, n, k, N, mode)
    assert B.ozaki2_cgemm(m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == 0
    torch.cuda.synchronize()
    got = np.asfortranarray(Cd.cpu().numpy().T)
    want = O.cgemm(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin[:m])
    assert got.dtype == np.complex64 and np.array_equal(got[:m], want)
    assert np.array_equal(got[m:], Cin[m:])
    if mode != 1 and N >= 9:
        ref = A.astype(np.complex128) @ Bm.astype(np.complex128)
        assert np.max(np.abs(O.cgemm(A, Bm, N, mode) - ref) / np.abs(ref)) < 1e-3


def test_cgemm_quick_returns_and_errors(B):
    import torch
    m, n, k, N = 32, 16, 24, 8
    A, Bm = _complex_inputs(m, n, k, 0.5, 5)
    Ad = torch.from_numpy(np.ascontiguousarray(A.astype(np.complex64).T)).cuda()
    Bd = torch.from_numpy(np.ascontiguousarray(Bm.astype(np.complex64).T)).cuda()
    Cin = np.asfortranarray((np.arange(m * n).reshape(m, n) * (1.0 + 0.5j)).astype(np.complex64))
    Cd = torch.from_numpy(np.ascontiguousarray(Cin.T)).cuda()
    B.ensure_zgemm_workspace(m, n, k, N, 2)
    assert B.ozaki2_cgemm(m, n, k, 0.0, Ad, m, Bd, k, 2.0j, Cd, m, N, 2) == 0        # alpha == 0: C := beta C
    torch.cuda.synchronize()
    assert np.array_equal(np.asfortranarray(Cd.cpu().numpy().T), (np.complex64(2.0j) * Cin).astype(np.complex64))
    assert B.ozaki2_cgemm(m, n, 0, 1.0, Ad, m, Bd, 1, 0.0, Cd, m, N, 2) == 0          # k == 0, beta == 0: zeros
    torch.cuda.synchronize()
    assert not np.any(Cd.cpu().numpy())
    assert B.ozaki2_cgemm(m, -1, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == -2
    assert B.ozaki2_cgemm(m, n, k, 1.0, Ad, m, Bd, k - 1, 0.0, Cd, m, N, 2) == -9
    assert B.ozaki2_cgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 5) == -15
    assert B.ozaki2_set_workspace(None, 0) == 0
    assert B.ozaki2_cgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == B.OZAKI2_ERR_WORKSPACE


def test_per_call_workspaces_on_concurrent_streams(B):
    # ozaki2_dgemm_ws / ozaki2_sgemm_ws: each call brings its own workspace, so calls on different streams are independent
    # (no registered workspace is needed or touched); several rounds enqueued without any synchronisation in between
    import torch
    assert B.ozaki2_set_workspace(None, 0) == 0
    probs = [(200, 136, 520, 14, 2, False), (129, 257, 1000, 17, 1, False), (96, 80, 300, 8, 2, True), (260, 40, 2049, 16, 0, False)]
    streams = [torch.cuda.Stream() for _ in probs]
    state = []
    for (m, n, k, N, mode, f32), st in zip(probs, streams):
        A, Bm = W.eq15_matrices(m, n, k, 1.0, 4000 + m + k)
        dt = np.float32 if f32 else np.float64
        A, Bm = np.asfortranarray(A.astype(dt)), np.asfortranarray(Bm.astype(dt))
        Ad = torch.from_numpy(np.ascontiguousarray(A.T)).cuda()
        Bd = torch.from_numpy(np.ascontiguousarray(Bm.T)).cuda()
        Cd = torch.full((n, m), float("nan"), dtype=Ad.dtype, device="cuda")
        nbytes = B.ozaki2_workspace_bytes(m, n, k, N, mode)
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        off = (-ws.data_ptr()) % 256
        state.append((A, Bm, Ad, Bd, Cd, ws, ws.data_ptr() + off, nbytes))
    torch.cuda.synchronize()
    for _ in range(3):
        for (m, n, k, N, mode, f32), st, (A, Bm, Ad, Bd, Cd, ws, wp, nbytes) in zip(probs, streams, state):
            fn = B.ozaki2_sgemm_ws if f32 else B.ozaki2_dgemm_ws
            assert fn(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, wp, nbytes, stream=st.cuda_stream) == 0
    torch.cuda.synchronize()
    for (m, n, k, N, mode, f32), (A, Bm, Ad, Bd, Cd, ws, wp, nbytes) in zip(probs, state):
        want = (O.sgemm if f32 else O.dgemm)(A, Bm, N, mode)
        assert np.array_equal(Cd.cpu().numpy().T, want), (m, n, k, N, mode, f32)
    # argument checks of the workspace itself: missing, too small, misaligned
    m, n, k, N, mode, _ = probs[0]
    A, Bm, Ad, Bd, Cd, ws, wp, nbytes = state[0]
    assert B.ozaki2_dgemm_ws(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, None, nbytes) == -14
    assert B.ozaki2_dgemm_ws(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, wp, nbytes - 1) == -14
    assert B.ozaki2_dgemm_ws(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode, wp + 8, nbytes) == -14
    assert B.ozaki2_dgemm_ws(m, n, k, 1.0, Ad, m - 1, Bd, k, 0.0, Cd, m, N, mode, wp, nbytes) == -6
    # the plain entry still reports the unregistered device workspace in its own way
    assert B.ozaki2_dgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, mode) == B.OZAKI2_ERR_WORKSPACE


def test_plain_launches_give_the_same_results(B):
    # OZAKI2_PDL=0 (read once per process) launches every kernel without the programmatic-launch attribute: same results
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, OZAKI2_PDL="0")
    r = subprocess.run([sys.executable, os.path.join(root, "__graft_entry__.py"), "--smoke"], env=env, capture_output=True, text=True,
                       timeout=600, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "smoke ok" in r.stdout


def test_row_major_call_with_the_workspace_the_query_reports(B):
    # the layout is not symmetric in m and n and a row-major call runs as the (n, m, k) problem: ozaki2_blas_workspace_bytes
    # reports what the call with that layout needs, and a workspace of exactly that size serves it (m = 300, n = 1: a
    # row-major call needs more than ozaki2_workspace_bytes(m, n, k) says)
    import torch
    m, n, k, N, mode = 300, 1, 64, 14, 2
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 31337)
    assert B.ozaki2_blas_workspace_bytes("C", m, n, k, N, mode) == B.ozaki2_workspace_bytes(m, n, k, N, mode)
    assert B.ozaki2_blas_workspace_bytes("R", m, n, k, N, mode) == B.ozaki2_workspace_bytes(n, m, k, N, mode)
    assert B.ozaki2_blas_workspace_bytes(101, m, n, k, N, mode) > B.ozaki2_blas_workspace_bytes(102, m, n, k, N, mode)
    want = O.dgemm(A, Bm, N, mode)
    for layout in ("R", "C"):
        need = B.ozaki2_blas_workspace_bytes(layout, m, n, k, N, mode)
        ws = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
        off = (-ws.data_ptr()) % 256
        assert B.ozaki2_set_workspace(ws.data_ptr() + off, need) == 0
        a = np.ascontiguousarray(A) if layout == "R" else np.ascontiguousarray(A.T)      # stored buffers, row by row
        b = np.ascontiguousarray(Bm) if layout == "R" else np.ascontiguousarray(Bm.T)
        Ad, Bd = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        Cd = torch.empty((m, n) if layout == "R" else (n, m), dtype=torch.float64, device="cuda")
        lda, ldb, ldc = (k, n, n) if layout == "R" else (m, k, m)
        assert B.ozaki2_dgemm_blas(layout, "N", "N", m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, ldc, N, mode) == 0
        torch.cuda.synchronize()
        got = Cd.cpu().numpy() if layout == "R" else Cd.cpu().numpy().T
        assert np.array_equal(got, want), layout
        assert B.ozaki2_set_workspace(None, 0) == 0
        del ws


def test_blas_entry_fuzz(B):
    # 36 seeded random problems through the BLAS-shaped entries: random layout, transposes, precision, shape (1 .. 300, k up
    # to 1500), N, mode, alpha / beta, leading-dimension padding and operand scales -- bit-exact against the oracle on the
    # logical matrices
    import torch
    rng = np.random.Generator(np.random.PCG64(20261106))
    for t in range(36):
        f32 = bool(rng.integers(0, 2))
        dt = np.float32 if f32 else np.float64
        m, n, k = int(rng.integers(1, 301)), int(rng.integers(1, 301)), int(rng.integers(1, 1501))
        N = int(rng.integers(2, 13)) if f32 else int(rng.integers(2, 21))
        mode = int(rng.integers(0, 3))
        rm, tra, trb = bool(rng.integers(0, 2)), bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
        alpha = float(rng.choice([1.0, -1.0, 0.5, 3.0]))
        beta = float(rng.choice([0.0, 1.0, -0.25]))
        sa, sb = (int(rng.integers(-20, 21)), int(rng.integers(-20, 21))) if f32 else (int(rng.integers(-200, 201)), int(rng.integers(-200, 201)))
        A, Bm = W.eq15_matrices(m, n, k, float(rng.uniform(0.0, 2.0)), 88000 + t)
        A, Bm = np.asfortranarray(np.ldexp(A, sa).astype(dt)), np.asfortranarray(np.ldexp(Bm, sb).astype(dt))
        Cin = rng.standard_normal((m, n)).astype(dt)
        bufA, lda = _stored(A, tra, rm, int(rng.integers(0, 4)))
        bufB, ldb = _stored(Bm, trb, rm, int(rng.integers(0, 4)))
        bufC, ldc = _stored(Cin, False, rm, int(rng.integers(0, 4)))
        Ad, Bd, Cd = torch.from_numpy(bufA).cuda(), torch.from_numpy(bufB).cuda(), torch.from_numpy(bufC.copy()).cuda()
        B.ensure_workspace(max(m, n), max(m, n), k, N, mode)
        call = B.ozaki2_sgemm_blas if f32 else B.ozaki2_dgemm_blas
        tag = f"fuzz {t}: f32={f32} {m}x{n}x{k} N{N} mode{mode} rm={rm} ta={tra} tb={trb} alpha={alpha} beta={beta}"
        assert call("R" if rm else "C", "T" if tra else "N", "T" if trb else "N", m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, mode) == 0, tag
        torch.cuda.synchronize()
        got = Cd.cpu().numpy()
        got = got[:, :n] if rm else got[:, :m].T
        with np.errstate(all="ignore"):
            want = (O.sgemm if f32 else O.dgemm)(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin.copy())
        assert np.array_equal(got, want, equal_nan=True), tag
