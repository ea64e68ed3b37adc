"""GPU parity of the SGEMM variant (-m gpu): ozaki2_sgemm against the oracle's sgemm, bit for bit (integer stages and
the FP32 result), on ragged shapes, every word count of P, wide-exponent FP32 inputs, alpha / beta."""
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


def f32_inputs(m, n, k, phi, seed):
    A, Bm = W.eq15_matrices(m, n, k, phi, seed)
    return np.asfortranarray(A.astype(np.float32)), np.asfortranarray(Bm.astype(np.float32))


@pytest.mark.parametrize("m,n,k,N,mode", [
    (200, 77, 333, 8, 2), (1, 1, 1, 2, 2), (129, 257, 127, 5, 1), (37, 300, 1000, 10, 0), (130, 40, 129, 12, 2),
    (300, 5, 31, 3, 0), (260, 260, 100, 6, 2), (64, 513, 260, 16, 2), (96, 96, 96, 20, 0), (513, 130, 4097, 9, 2),
])
def test_sgemm_all_stages_bit_exact(B, m, n, k, N, mode):
    import torch
    A, Bm = f32_inputs(m, n, k, 1.0, 500 + m + n + k + N)
    Ad, Bd = B.colmajor_to_device(A, np.float32), B.colmajor_to_device(Bm, np.float32)
    g = B.dgemm_stages(Ad, Bd, N, mode, want=("e", "f", "resA", "resB", "U", "Cpp"))
    torch.cuda.synchronize()
    o = O.stages(A.astype(np.float64), Bm.astype(np.float64), N, mode)      # integer stages = FP64 path on promoted inputs
    assert np.array_equal(g["e"].cpu().numpy(), o["e"]) and np.array_equal(g["f"].cpu().numpy(), o["f"])
    assert np.array_equal(g["resA"].cpu().numpy(), o["RA"]) and np.array_equal(g["resB"].cpu().numpy(), o["RB"])
    assert np.array_equal(g["U"].cpu().numpy(), o["U"])
    assert np.array_equal(g["Cpp"].cpu().numpy().view(np.uint64), o["Cpp"])
    Cg = B.device_to_colmajor(g["C"])
    assert Cg.dtype == np.float32
    assert np.array_equal(Cg, O.sgemm(A, Bm, N, mode))


def test_sgemm_alpha_beta_ld_and_quick_returns(B):
    import torch
    m, n, k, N = 70, 50, 90, 8
    A, Bm = f32_inputs(m, n, k, 0.5, 21)
    lda, ldb, ldc = m + 3, k + 5, m + 7
    Ap = np.zeros((lda, k), np.float32, order="F"); Ap[:m] = A
    Bp = np.zeros((ldb, n), np.float32, order="F"); Bp[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(3))
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)).astype(np.float32))
    Ad, Bd = B.colmajor_to_device(Ap, np.float32), B.colmajor_to_device(Bp, np.float32)
    B.ensure_workspace(m, n, k, N, 2)
    for alpha, beta in ((0.7, -1.3), (1.0, 0.0), (-2.0, 1.0), (0.0, 0.5), (0.0, 0.0)):
        Cd = B.colmajor_to_device(Cin, np.float32)
        assert B.ozaki2_sgemm(m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, 2) == 0
        torch.cuda.synchronize()
        got = B.device_to_colmajor(Cd)
        if alpha == 0.0:
            want = np.zeros((m, n), np.float32) if beta == 0.0 else (np.float32(beta) * Cin[:m]).astype(np.float32)
        else:
            want = O.sgemm(A, Bm, N, 2, alpha=alpha, beta=beta, C_in=Cin[:m].copy())
        assert np.array_equal(got[:m], want), (alpha, beta)
        assert np.array_equal(got[m:], Cin[m:])


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_sgemm_wide_exponent_fp32_inputs(B, mode):
    # exponents over the whole FP32 range (normal and subnormal), zeros, a zero row and a zero column
    import torch
    rng = np.random.Generator(np.random.PCG64(17))

    def one(rows, cols):
        v = (rng.random(rows * cols) + 1.0) * np.exp2(rng.integers(-148, 60, size=rows * cols)) * (rng.integers(0, 2, size=rows * cols) * 2 - 1)
        v[rng.random(rows * cols) < 0.05] = 0.0
        return v.astype(np.float32).reshape(cols, rows).T.copy()

    A, Bm = one(140, 200), one(200, 70)
    A[70, :] = 0.0
    Bm[:, 23] = 0.0
    A[3, :] = np.float32(1e-45)
    A, Bm = np.asfortranarray(A), np.asfortranarray(Bm)
    Ad, Bd = B.colmajor_to_device(A, np.float32), B.colmajor_to_device(Bm, np.float32)
    g = B.dgemm_stages(Ad, Bd, 10, mode, want=("e", "f", "Cpp"))
    torch.cuda.synchronize()
    Co, eo, fo = O.sgemm(A, Bm, 10, mode, return_exponents=True)
    assert np.array_equal(g["e"].cpu().numpy(), eo) and np.array_equal(g["f"].cpu().numpy(), fo)
    assert np.array_equal(B.device_to_colmajor(g["C"]), Co)
