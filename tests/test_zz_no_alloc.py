"""ozaki2_row_exponents_noalloc -- the one call of the library that needs no workspace.

Everything else in libozaki2 works in a workspace that the caller has to allocate on the device.  That is not
always possible: a plug-in inside an application that reserved the whole GPU for its own memory pool cannot get
more from cudaMalloc, and code on a latency-critical path may not call cudaMalloc / cudaFree at all because they
stall every stream of the device.  For such callers the library carries a fixed 1 MiB scratch array in its own
image (room for OZAKI2_NOALLOC_MAX_ROWS = 65536 rows) and this entry point computes the row scaling exponents of A
with it; only the input A and the output e come from the caller.

What is checked: the exponents equal, bit for bit (the bar of every integer stage in this repository), the `e` of
the existing workspace path (ozaki2_dgemm_stages) -- on two calls in a row with different matrices, because all calls
share the one array and the second call finds the first call's statistics in it -- and the size limit is refused
with its own error code.

The file name keeps this module last in pytest's collection order: under `pytest -x` a failure here cannot hide
another test.  It depends on no other test having run (or not run) before it.
"""
import numpy as np
import pytest

import workloads as W


@pytest.fixture(scope="module")
def B():
    import paper_2606_29129_b200 as pkg
    pkg.lib()                       # fails loudly if libozaki2.so is missing
    return pkg


def test_rows_beyond_the_builtin_scratch_are_refused(B):
    """More rows than the static array has room for: a dedicated status, a message that names the limit, nothing launched
    (the pointers here are never dereferenced, so this runs without a GPU)."""
    before = B.ozaki2_kernel_launches()
    m = B.OZAKI2_NOALLOC_MAX_ROWS + 1
    rc = B.ozaki2_row_exponents_noalloc(m, 64, 256, m, 14, B.OZAKI2_MODE_PROP, 256, stream=0)
    assert rc == B.OZAKI2_ERR_NOALLOC_LIMIT
    assert "OZAKI2_NOALLOC_MAX_ROWS" in B.ozaki2_status_string(rc)
    # the ordinary argument checks, numbered by position in the prototype
    assert B.ozaki2_row_exponents_noalloc(-1, 64, 256, 1, 14, 2, 256, stream=0) == -1
    assert B.ozaki2_row_exponents_noalloc(8, -1, 256, 8, 14, 2, 256, stream=0) == -2
    assert B.ozaki2_row_exponents_noalloc(8, 64, None, 8, 14, 2, 256, stream=0) == -3
    assert B.ozaki2_row_exponents_noalloc(8, 64, 256, 7, 14, 2, 256, stream=0) == -4
    assert B.ozaki2_row_exponents_noalloc(8, 64, 256, 8, 21, 2, 256, stream=0) == -5
    assert B.ozaki2_row_exponents_noalloc(8, 64, 256, 8, 14, B.OZAKI2_MODE_ACCURATE, 256, stream=0) == -6
    assert B.ozaki2_row_exponents_noalloc(8, 64, 256, 8, 14, 2, None, stream=0) == -7
    assert B.ozaki2_row_exponents_noalloc(0, 64, None, 1, 14, 2, None, stream=0) == 0
    assert B.ozaki2_kernel_launches() == before


def _existing_path_e(B, A, N, mode):
    """e of the workspace path: ozaki2_dgemm_stages on (A, some B); e_i depends on row i of A only."""
    import torch
    m, k = A.shape
    _, Bm = W.eq15_matrices(1, 8, k, 0.5, 4242)
    out = B.dgemm_stages(B.colmajor_to_device(A), B.colmajor_to_device(Bm), N, mode, want=("e",))
    torch.cuda.synchronize()
    return out["e"].cpu().numpy()


def _noalloc_e(B, A_dev, m, k, lda, N, mode, e_dev):
    rc = B.ozaki2_row_exponents_noalloc(m, k, A_dev, lda, N, mode, e_dev)
    assert rc == 0, B.ozaki2_status_string(rc)


@pytest.mark.gpu
@pytest.mark.parametrize("mode", [2, 1])
def test_two_calls_in_a_row_match_the_workspace_path(B, mode):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    N = 16
    # call 1: several row blocks and k slices, ragged in both directions, entries spread over many binades
    m1, k1 = 1100, 1500
    A1, _ = W.eq15_matrices(m1, 1, k1, 2.0, 77001 + mode)
    A1[5, :] = 0.0                                     # an all-zero row: exponent 0
    A1[6, :] *= 2.0 ** -1040                           # a row of subnormals: the exact-pattern branch
    A1[7, :] *= 2.0 ** 900
    # call 2: fewer rows, another k, much smaller magnitudes -- statistics left over from call 1 (larger maxima,
    # non-zero sums) would change these exponents if the call did not clear its part of the shared array
    m2, k2 = 333, 900
    A2, _ = W.eq15_matrices(m2, 1, k2, 0.5, 77011 + mode)
    A2 *= 2.0 ** -60
    A2[0, :] = 0.0
    want1, want2 = _existing_path_e(B, A1, N, mode), _existing_path_e(B, A2, N, mode)
    assert want1[5] == 0 and want2[0] == 0 and len(set(want1.tolist())) > 3

    lda1 = m1 + 3                                      # padded leading dimension
    A1d = torch.zeros((k1, lda1), dtype=torch.float64, device="cuda")
    A1d[:, :m1] = torch.from_numpy(np.ascontiguousarray(A1.T)).cuda()
    A2d = B.colmajor_to_device(A2)
    e1 = torch.full((m1 + 8,), -12345, dtype=torch.int32, device="cuda")
    e2 = torch.full((m2 + 8,), -12345, dtype=torch.int32, device="cuda")
    launches = B.ozaki2_kernel_launches()
    _noalloc_e(B, A1d, m1, k1, lda1, N, mode, e1)      # same stream, back to back: stream order is the only ordering
    _noalloc_e(B, A2d, m2, k2, m2, N, mode, e2)
    torch.cuda.synchronize()
    assert B.ozaki2_kernel_launches() - launches == 6   # three kernels a call; the library's kernels, not a fallback
    assert np.array_equal(e1[:m1].cpu().numpy(), want1)
    assert np.array_equal(e2[:m2].cpu().numpy(), want2)
    assert (e1[m1:] == -12345).all() and (e2[m2:] == -12345).all()      # nothing written past e[m)
    # and once more the first problem, now on top of the second one's leftovers
    e1.fill_(-12345)
    _noalloc_e(B, A1d, m1, k1, lda1, N, mode, e1)
    torch.cuda.synchronize()
    assert np.array_equal(e1[:m1].cpu().numpy(), want1)


@pytest.mark.gpu
def test_empty_rows_and_the_largest_row_count(B):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    # k == 0: every row is empty, exponent 0
    e = torch.full((40,), 7, dtype=torch.int32, device="cuda")
    assert B.ozaki2_row_exponents_noalloc(40, 0, None, 40, 14, 2, e) == 0
    torch.cuda.synchronize()
    assert (e == 0).all()
    # the full array: OZAKI2_NOALLOC_MAX_ROWS rows, short k
    m, k, N = B.OZAKI2_NOALLOC_MAX_ROWS, 40, 14
    A, _ = W.eq15_matrices(m, 1, k, 1.0, 77100)
    want = _existing_path_e(B, A, N, 2)
    Ad = B.colmajor_to_device(A)
    e = torch.empty((m,), dtype=torch.int32, device="cuda")
    _noalloc_e(B, Ad, m, k, m, N, 2, e)
    torch.cuda.synchronize()
    assert np.array_equal(e.cpu().numpy(), want)
