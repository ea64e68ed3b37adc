"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded inputs, element by element.

Bar (BASELINE.json north_star): bit-exact on every integer stage -- scaling exponents, INT8 residues,
per-modulus products mod p_l, the recovered integer C'' -- and max elementwise relative difference
<= 2^-50 on the final FP64 C.  With alpha = 1, beta = 0 the final C is in fact required bit-identical here
(C = RN(C'') 2^-(e+f) has a single rounding on both sides).
"""
import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O

pytestmark = pytest.mark.gpu

TOL_C = 2.0 ** -50


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_29129_b200 as pkg
    pkg.lib()                       # fails loudly if libozaki2.so is missing
    return pkg


def gpu_stages(B, A, Bm, N, mode, **kw):
    import torch
    Ad, Bd = B.colmajor_to_device(A), B.colmajor_to_device(Bm)
    want = ["e", "f", "resA", "resB", "U", "Cpp"] + (["rowmax", "colmax"] if mode == 0 else [])
    out = B.dgemm_stages(Ad, Bd, N, mode, want=want, **kw)
    torch.cuda.synchronize()
    res = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in out.items()}
    res["C"] = np.asfortranarray(res["C"].T)
    res["Cpp"] = res["Cpp"].view(np.uint64)
    return res


def assert_stage_parity(g, o, mode, tag=""):
    assert np.array_equal(g["e"], o["e"]), f"{tag} e"
    assert np.array_equal(g["f"], o["f"]), f"{tag} f"
    if mode == 0:
        assert np.array_equal(g["rowmax"].astype(np.int64), o["rowmax"]), f"{tag} rowmax"
        assert np.array_equal(g["colmax"].astype(np.int64), o["colmax"]), f"{tag} colmax"
    assert np.array_equal(g["resA"], o["RA"]), f"{tag} resA"
    assert np.array_equal(g["resB"], o["RB"]), f"{tag} resB"
    assert np.array_equal(g["U"], o["U"]), f"{tag} U"
    assert np.array_equal(g["Cpp"], o["Cpp"]), f"{tag} C''"
    assert np.array_equal(g["C"], o["C"]), f"{tag} C"
    nz = o["C"] != 0
    if nz.any():
        assert np.max(np.abs(g["C"][nz] - o["C"][nz]) / np.abs(o["C"][nz])) <= TOL_C


# --------------------------------------------------------------------------------------------- config 0
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_config0_128_all_stages(B, mode):
    A, Bm = W.config_matrices(0)
    N = 14
    o = O.stages(A, Bm, N, mode, want_exact=True)
    g = gpu_stages(B, A, Bm, N, mode)
    assert_stage_parity(g, o, mode, f"cfg0 mode{mode}")
    # and against the exact __int128-style product: C'' == A'B' whenever |A'B'| < P/2 (always here)
    assert o["counts"]["wrong"] == 0
    assert np.array_equal(g["Cpp"], o["Z"])


# --------------------------------------------------------------------------------------------- ragged shapes, all N
@pytest.mark.parametrize("m,n,k,N,mode", [
    (200, 77, 333, 14, 2), (1, 1, 1, 2, 2), (129, 257, 127, 9, 1), (37, 300, 1000, 16, 0), (130, 40, 129, 17, 2),
    (64, 513, 260, 20, 0), (255, 255, 4097, 20, 2), (16, 16, 16, 3, 1), (300, 5, 31, 15, 0), (5, 300, 2049, 8, 2),
    (260, 260, 100, 12, 2), (128, 256, 128, 4, 2), (131, 100, 777, 5, 0), (100, 131, 64, 18, 1), (77, 77, 77, 13, 2),
    (33, 65, 640, 6, 2), (90, 70, 50, 7, 1), (48, 40, 131072, 14, 2), (40, 24, 131072, 20, 0),
    (40, 24, (1 << 18) + 384, 14, 2), (24, 40, (1 << 18) + 129, 16, 1), (130, 20, 1 << 18, 15, 0), (70, 90, 150, 10, 0), (50, 60, 70, 11, 2), (61, 67, 71, 19, 0),
])
def test_ragged_shapes_and_every_moduli_count(B, m, n, k, N, mode):
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 1000 + m + n + k + N)
    o = O.stages(A, Bm, N, mode)
    g = gpu_stages(B, A, Bm, N, mode)
    assert_stage_parity(g, o, mode, f"{m}x{n}x{k} N{N} mode{mode}")


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("N", [14, 20])
def test_wide_exponent_inputs_zero_rows_subnormals(B, mode, N):
    A, Bm = W.wide_exponent_matrices(140, 70, 200, seed=7 + N)
    A[3, :] = np.ldexp(1.0, -1074)
    A[4, :5] = 5e-324
    o = O.stages(A, Bm, N, mode)
    g = gpu_stages(B, A, Bm, N, mode)
    assert_stage_parity(g, o, mode, f"wide N{N} mode{mode}")


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_structured_inputs(B, mode):
    for A, Bm in (W.all_ones_scaled(130, 60, 256, 2.0 ** -4), W.small_integer_matrices(50, 40, 300, 8, 5),
                  (np.asfortranarray(np.eye(64)), W.eq15_matrices(64, 32, 64, 2.0, 3)[1])):
        o = O.stages(A, Bm, 20, mode)
        g = gpu_stages(B, A, Bm, 20, mode)
        assert_stage_parity(g, o, mode, "structured")


# --------------------------------------------------------------------------------------------- alpha / beta, lda
def test_alpha_beta_and_leading_dimensions(B):
    import torch
    m, n, k, N = 70, 50, 90, 14
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 77)
    lda, ldb, ldc = m + 3, k + 5, m + 7
    Ap = np.zeros((lda, k), order="F"); Ap[:m] = A
    Bp = np.zeros((ldb, n), order="F"); Bp[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(3))
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)))
    Ad, Bd, Cd = B.colmajor_to_device(Ap), B.colmajor_to_device(Bp), B.colmajor_to_device(Cin)
    B.ensure_workspace(m, n, k, N, 2)
    for alpha, beta in ((0.7, -1.3), (1.0, 0.0), (-2.0, 1.0), (0.0, 0.5), (0.0, 0.0)):
        Cd.copy_(B.colmajor_to_device(Cin))
        rc = B.ozaki2_dgemm(m, n, k, alpha, Ad, lda, Bd, ldb, beta, Cd, ldc, N, 2)
        assert rc == 0
        torch.cuda.synchronize()
        got = B.device_to_colmajor(Cd)
        if alpha == 0.0:
            want = np.zeros((m, n)) if beta == 0.0 else beta * Cin[:m]
        else:
            want = O.dgemm(A, Bm, N, 2, alpha=alpha, beta=beta, C_in=Cin[:m].copy())
        assert np.array_equal(got[:m], want), (alpha, beta)
        assert np.array_equal(got[m:], Cin[m:])               # rows beyond m untouched
    # beta == 0 must overwrite NaNs (BLAS rule)
    Cd.fill_(float("nan"))
    assert B.ozaki2_dgemm(m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, ldc, N, 2) == 0
    torch.cuda.synchronize()
    assert np.array_equal(B.device_to_colmajor(Cd)[:m], O.dgemm(A, Bm, N, 2))


def test_workspace_errors(B):
    import torch
    A, Bm = W.eq15_matrices(64, 64, 64, 0.5, 1)
    Ad, Bd = B.colmajor_to_device(A), B.colmajor_to_device(Bm)
    Cd = torch.empty((64, 64), dtype=torch.float64, device="cuda")
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    assert B.ozaki2_set_workspace(small, small.numel()) == 0
    assert B.ozaki2_dgemm(64, 64, 64, 1.0, Ad, 64, Bd, 64, 0.0, Cd, 64, 14, 2) == B.OZAKI2_ERR_WORKSPACE
    assert B.ozaki2_set_workspace(None, 0) == 0
    assert B.ozaki2_dgemm(64, 64, 64, 1.0, Ad, 64, Bd, 64, 0.0, Cd, 64, 14, 2) == B.OZAKI2_ERR_WORKSPACE
    B.ensure_workspace(64, 64, 64, 14, 2)
    assert B.ozaki2_dgemm(64, 64, 64, 1.0, Ad, 64, Bd, 64, 0.0, Cd, 64, 14, 2) == 0
    torch.cuda.synchronize()


def test_host_buffer_entry_point(B):
    import torch
    m, n, k, N = 96, 80, 200, 15
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 5)
    B.ensure_workspace(m, n, k, N, 2)
    nbytes = B.ozaki2_host_scratch_bytes(m, n, k)
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    Ch = np.zeros((m, n), order="F")
    rc = B.ozaki2_dgemm_host(m, n, k, 1.0, A, m, Bm, k, 0.0, Ch, m, N, 2, scratch, nbytes)
    assert rc == 0
    assert np.array_equal(Ch, O.dgemm(A, Bm, N, 2))


@pytest.mark.parametrize("mode,alpha,beta", [(2, 1.0, 0.0), (1, -0.5, 2.0), (0, 1.0, 0.0)])
def test_host_buffer_entry_point_column_panels(B, mode, alpha, beta):
    # n >= 512: modes 1, 2 run as column panels with the copies overlapped (5 panels here, the last one ragged);
    # padded leading dimensions on all three host matrices
    import torch
    m, n, k, N = 300, 1100, 200, 14
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 6)
    lda, ldb, ldc = m + 4, k + 2, m + 6
    Ah = np.zeros((lda, k), order="F"); Ah[:m] = A
    Bh = np.zeros((ldb, n), order="F"); Bh[:k] = Bm
    rng = np.random.Generator(np.random.PCG64(4))
    Cin = np.asfortranarray(rng.standard_normal((ldc, n)))
    Ch = Cin.copy(order="F")
    B.ensure_workspace(m, n, k, N, mode)
    nbytes = B.ozaki2_host_scratch_bytes(m, n, k)
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    rc = B.ozaki2_dgemm_host(m, n, k, alpha, Ah, lda, Bh, ldb, beta, Ch, ldc, N, mode, scratch, nbytes)
    assert rc == 0
    want = O.dgemm(A, Bm, N, mode, alpha=alpha, beta=beta, C_in=Cin[:m].copy())
    assert np.array_equal(Ch[:m], want)
    assert np.array_equal(Ch[m:], Cin[m:])


@pytest.mark.parametrize("transa,transb", [(0, 0), (1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_transposed_operands(B, transa, transb, mode):
    # the stored matrices are op(X)^T with padded leading dimensions; the result must be the oracle's on the logical A, B
    import torch
    m, n, k, N = 150, 90, 260, 15
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 321)
    SA = A.T if transa else A                                # stored A: k x m or m x k
    SB = Bm.T if transb else Bm                              # stored B: n x k or k x n
    lda, ldb = SA.shape[0] + 3, SB.shape[0] + 5
    PA = np.zeros((lda, SA.shape[1]), order="F"); PA[:SA.shape[0]] = SA
    PB = np.zeros((ldb, SB.shape[1]), order="F"); PB[:SB.shape[0]] = SB
    Ad, Bd = B.colmajor_to_device(PA), B.colmajor_to_device(PB)
    Cd = torch.full((n, m), float("nan"), dtype=torch.float64, device="cuda")
    B.ensure_workspace(m, n, k, N, mode)
    assert B.ozaki2_dgemm_t(transa, transb, m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, m, N, mode) == 0
    torch.cuda.synchronize()
    assert np.array_equal(B.device_to_colmajor(Cd), O.dgemm(A, Bm, N, mode))
    assert B.ozaki2_dgemm_t(2, 0, m, n, k, 1.0, Ad, lda, Bd, ldb, 0.0, Cd, m, N, mode) == -1
    assert B.ozaki2_dgemm_t(transa, transb, m, n, k, 1.0, Ad, SA.shape[0] - 1, Bd, ldb, 0.0, Cd, m, N, mode) == -8


@pytest.mark.parametrize("mode", [1, 2])
def test_non_finite_inputs_stay_in_their_row_and_column(B, mode):
    # include/ozaki2.h: Inf / NaN are not detected; they may spoil their own row of A / column of B only (in the
    # fast modes e_i, f_j and the residues are row / column local) and never hang or fault
    import torch
    m, n, k, N = 96, 80, 300, 14
    A, Bm = W.eq15_matrices(m, n, k, 0.5, 42)
    Ad, Bd = B.colmajor_to_device(A), B.colmajor_to_device(Bm)
    clean = B.device_to_colmajor(B.dgemm(Ad, Bd, N, mode))
    A2, B2 = A.copy(order="F"), Bm.copy(order="F")
    A2[3, 7] = np.nan; A2[10, 0] = np.inf; B2[5, 9] = -np.inf; B2[100, 33] = np.nan
    dirty = B.device_to_colmajor(B.dgemm(B.colmajor_to_device(A2), B.colmajor_to_device(B2), N, mode))
    torch.cuda.synchronize()
    rows = np.ones(m, bool); rows[[3, 10]] = False
    cols = np.ones(n, bool); cols[[9, 33]] = False
    assert np.array_equal(dirty[np.ix_(rows, cols)], clean[np.ix_(rows, cols)])


def test_call_is_cuda_graph_capturable(B):
    # "CUDA streams and graphs": after the first call on a device (which uploads the constant tables) the path only
    # enqueues kernels and memsets on the caller's stream, so it can be captured and replayed
    import torch
    m, n, k, N = 256, 192, 320, 14
    A, Bm = W.eq15_matrices(m, n, k, 0.5, 12)
    Ad, Bd = B.colmajor_to_device(A), B.colmajor_to_device(Bm)
    Cd = torch.empty((n, m), dtype=torch.float64, device="cuda")
    B.ensure_workspace(m, n, k, N, 2)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        assert B.ozaki2_dgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == 0
    torch.cuda.synchronize()
    want = O.dgemm(A, Bm, N, 2)
    assert np.array_equal(B.device_to_colmajor(Cd), want)
    g = torch.cuda.CUDAGraph()
    Cd.zero_()
    with torch.cuda.graph(g):
        assert B.ozaki2_dgemm(m, n, k, 1.0, Ad, m, Bd, k, 0.0, Cd, m, N, 2) == 0
    for _ in range(3):
        Cd.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(B.device_to_colmajor(Cd), want)


# --------------------------------------------------------------------------------------------- primitives
def test_log2f_exhaustive_equals_oracle(B):
    import torch
    bits = np.arange(0x3F800000, 0x40000000 + 1, dtype=np.uint32)
    x = bits.view(np.float32)
    xd = torch.from_numpy(x.copy()).cuda()
    yd = torch.empty_like(xd)
    assert B.ozaki2_debug_log2f(xd, yd, x.size) == 0
    torch.cuda.synchronize()
    assert np.array_equal(yd.cpu().numpy(), O.log2f_array(x))


def test_epilogue_mod_p_all_moduli(B):
    import torch
    rng = np.random.Generator(np.random.PCG64(9))
    v = np.concatenate([rng.integers(-2 ** 31, 2 ** 31, size=1 << 22, dtype=np.int64),
                        np.array([-2 ** 31, 2 ** 31 - 1, -1, 0, 1, 2 ** 16, -2 ** 16, 2 ** 16 - 1, 65535 * 32768], np.int64),
                        np.arange(-70000, 70000, dtype=np.int64)]).astype(np.int32)
    vd = torch.from_numpy(v).cuda()
    od = torch.empty(v.size, dtype=torch.uint8, device="cuda")
    p = O.constants(20)["p"]
    for l in range(20):
        assert B.ozaki2_debug_mod_p(l, vd, od, v.size) == 0
        torch.cuda.synchronize()
        assert np.array_equal(od.cpu().numpy(), (v.astype(np.int64) % p[l]).astype(np.uint8)), l


@pytest.mark.parametrize("m,n,k,N", [(128, 256, 128, 1), (256, 512, 1024, 3), (384, 272, 2048, 20), (16, 8, 128, 2),
                                     (1040, 784, 512, 5)])
def test_residue_gemm_tensor_core_vs_oracle_and_check_kernel(B, m, n, k, N):
    import torch
    rng = np.random.Generator(np.random.PCG64(k + N))
    p = O.constants(20)["p"][:N]
    RA = np.stack([rng.integers(-(q // 2), (q - 1) // 2 + 1, size=(m, k)) for q in p]).astype(np.int8)
    RB = np.stack([rng.integers(-(q // 2), (q - 1) // 2 + 1, size=(n, k)) for q in p]).astype(np.int8)
    want, _ = O.products(max(N, 2), RA if N > 1 else np.concatenate([RA, RA]), RB if N > 1 else np.concatenate([RB, RB]))
    want = want[:N]
    RAd, RBd = torch.from_numpy(RA).cuda(), torch.from_numpy(RB).cuda()
    for tc in (2, 1, 0):            # CTA pairs / one CTA per tile / CUDA-core check kernel
        Ud = torch.zeros((N, n, m), dtype=torch.uint8, device="cuda")
        assert B.ozaki2_debug_residue_gemm(N, m, n, k, RAd, RBd, Ud, tc) == 0
        torch.cuda.synchronize()
        assert np.array_equal(Ud.cpu().numpy(), want), f"tensor_cores={tc}"


def test_mma_only_variants_leave_U_untouched(B):
    # variants 3 / 4 of ozaki2_debug_residue_gemm (the INT8 ceiling runs of bench.py) hand the accumulator back unread
    import torch
    N, m, n, k = 2, 256, 512, 256
    RA = torch.randint(-100, 100, (N, m, k), dtype=torch.int8, device="cuda")
    RB = torch.randint(-100, 100, (N, n, k), dtype=torch.int8, device="cuda")
    Ud = torch.full((N, n, m), 7, dtype=torch.uint8, device="cuda")
    for variant in (3, 4):
        assert B.ozaki2_debug_residue_gemm(N, m, n, k, RA, RB, Ud, variant) == 0
        torch.cuda.synchronize()
        assert bool((Ud == 7).all())
    assert B.ozaki2_debug_residue_gemm(N, m, n, k, RA, RB, Ud, 5) == -8


def test_k_blocked_residue_gemm_beyond_2pow17(B):
    # k > 2^17 is computed in blocks of 2^17 whose residues are added mod p_l in the epilogue; worst-case
    # operands (-128 x -128 for p = 256, 127 x 127 for 255) over 2 1/2 blocks
    import torch
    m, n, k, N = 128, 256, (1 << 18) + (1 << 16), 3
    rng = np.random.Generator(np.random.PCG64(11))
    RA = np.zeros((N, m, k), np.int8); RB = np.zeros((N, n, k), np.int8)
    RA[0] = -128; RB[0] = -128
    RA[1] = 127; RB[1] = 127
    RA[2, :8] = rng.integers(-126, 127, size=(8, k)); RB[2, :8] = rng.integers(-126, 127, size=(8, k))
    want, _ = O.products(N, RA[:, :8], RB[:, :8])
    RAd, RBd = torch.from_numpy(RA).cuda(), torch.from_numpy(RB).cuda()
    Ud = torch.zeros((N, n, m), dtype=torch.uint8, device="cuda")
    assert B.ozaki2_debug_residue_gemm(N, m, n, k, RAd, RBd, Ud, 1) == 0
    torch.cuda.synchronize()
    got = Ud.cpu().numpy()
    assert np.array_equal(got[:, :8, :8], want)
    assert np.all(got[0] == (128 * 128 * k) % 256) and np.all(got[1] == (127 * 127 * k) % 255)


def test_int32_accumulator_wraps_at_k_2pow17(B):
    # reading R6: p = 256 residues of -128 over k = 2^17 give 2^31, which must WRAP (256 | 2^32), not saturate;
    # the odd moduli stay below 2^31.
    import torch
    m, n, k, N = 256, 256, 1 << 17, 2
    RA = np.zeros((N, m, k), np.int8)
    RB = np.zeros((N, n, k), np.int8)
    RA[0] = -128; RB[0] = -128
    RA[1] = 127; RB[1] = 127
    RA[0, 5, :7] = 3                      # make one row differ so that the result is not constant
    want, maxR = O.products(N, RA[:, :8], RB[:, :8])
    assert maxR == 2 ** 31
    RAd, RBd = torch.from_numpy(RA).cuda(), torch.from_numpy(RB).cuda()
    Ud = torch.zeros((N, n, m), dtype=torch.uint8, device="cuda")
    for tc in (1, 2):
        Ud.zero_()
        assert B.ozaki2_debug_residue_gemm(N, m, n, k, RAd, RBd, Ud, tc) == 0
        torch.cuda.synchronize()
        got = Ud.cpu().numpy()
        assert np.array_equal(got[:, :8, :8], want)
        assert np.all(got[1] == (127 * 127 * k) % 255)


@pytest.mark.parametrize("m,n,k,N,mode,phi", [
    (1500, 1301, 2101, 16, 2, 1.0),      # several waves of ragged tiles in every persistent kernel, k tail of 53
    (1031, 1540, 1667, 18, 0, 2.0),      # wide conversion format (N >= 17), five words of P, accurate mode's auxiliary product
    (2050, 515, 3073, 15, 1, 0.5),       # one row / column past a tile boundary, k = 24 x 128 + 1
])
def test_midsize_ragged_shapes_all_stages(B, m, n, k, N, mode, phi):
    # between the small ragged cases above (at most a wave of tiles) and the sampled full-size tests (tile-aligned shapes):
    # every stage compared in full on shapes whose persistent loops run many items with ragged edges in m, n and k
    A, Bm = W.eq15_matrices(m, n, k, phi, 5000 + m + n + k)
    o = O.stages(A, Bm, N, mode)
    g = gpu_stages(B, A, Bm, N, mode)
    assert_stage_parity(g, o, mode, f"{m}x{n}x{k} N{N} mode{mode}")
    # and the plain call (product kernels: crt_fast + hand-over instead of crt_exact for every element)
    import torch
    Cd = B.dgemm(B.colmajor_to_device(A), B.colmajor_to_device(Bm), N, mode)
    torch.cuda.synchronize()
    assert np.array_equal(B.device_to_colmajor(Cd), o["C"])


def test_random_shapes_fuzz(B):
    # 40 seeded random problems: shapes 1 .. 400 (k up to 3000), every N and mode, eq. (15) data with phi in [0, 4] and a
    # random power-of-two scale on each operand; all stages bit-exact
    rng = np.random.Generator(np.random.PCG64(20261105))
    for t in range(40):
        m, n = int(rng.integers(1, 401)), int(rng.integers(1, 401))
        k = int(rng.integers(1, 3001)) if t % 4 else int(rng.integers(1, 40))
        N, mode = int(rng.integers(2, 21)), int(rng.integers(0, 3))
        phi = float(rng.uniform(0.0, 4.0))
        sa, sb = int(rng.integers(-300, 301)), int(rng.integers(-300, 301))
        A, Bm = W.eq15_matrices(m, n, k, phi, 77000 + t)
        A, Bm = np.ldexp(A, sa), np.ldexp(Bm, sb)
        o = O.stages(A, Bm, N, mode)
        g = gpu_stages(B, A, Bm, N, mode)
        assert_stage_parity(g, o, mode, f"fuzz {t}: {m}x{n}x{k} N{N} mode{mode} phi{phi:.2f} 2^{sa} 2^{sb}")
