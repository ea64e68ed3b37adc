"""CPU-side checks of the C-ABI boundary: the library builds and loads, exports every symbol that
include/ozaki2.h declares, validates arguments (BLAS xerbla numbering) and reports its Step-1 constants.
No kernel is launched here (no GPU needed)."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest
from mpmath import mp, mpf, log

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    if not os.path.exists(os.path.join(ROOT, "paper_2606_29129_b200", "libozaki2.so")):
        subprocess.run([sys.executable, os.path.join(ROOT, "paper_2606_29129_b200", "build.py")], check=True)
    import paper_2606_29129_b200 as pkg
    pkg.lib()
    return pkg


def test_every_declared_symbol_is_exported(B):
    hdr = open(os.path.join(ROOT, "include", "ozaki2.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(ozaki2_[a-z0-9_]+)\s*\(", hdr))
    assert {"ozaki2_dgemm", "ozaki2_workspace_bytes", "ozaki2_set_workspace", "ozaki2_dgemm_host",
            "ozaki2_dgemm_stages", "ozaki2_get_constants", "ozaki2_status_string"} <= names
    L = B.lib()
    for nm in names:
        assert hasattr(L, nm), nm


def test_product_does_not_import_the_oracle():
    # the product path shares nothing with oracle/: no import, no include, no dlopen of it
    pat = re.compile(r"(^\s*(from|import)\s+oracle\b)|(#include\s*[<\"][^>\"]*oracle)|(libozaki2_oracle)", re.M)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2606_29129_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                assert not pat.search(open(os.path.join(dirpath, fn)).read()), fn


def test_argument_checks_xerbla_numbering(B):
    ok = dict(m=8, n=8, k=8, alpha=1.0, A=256, lda=8, B=256, ldb=8, beta=0.0, Cm=256, ldc=8, num_moduli=14, scaling_mode=2)

    def call(**kw):
        a = dict(ok, **kw)
        return B.ozaki2_dgemm(a["m"], a["n"], a["k"], a["alpha"], a["A"], a["lda"], a["B"], a["ldb"], a["beta"], a["Cm"],
                              a["ldc"], a["num_moduli"], a["scaling_mode"], stream=0)

    assert call(m=-1) == -1
    assert call(n=-1) == -2
    assert call(k=-1) == -3
    assert call(k=(1 << 22) + 1) == -3            # OZAKI2_MAX_K (blocked beyond 2^17)
    assert call(k=(1 << 18) + 1, scaling_mode=0) == -3   # accurate mode: auxiliary product must fit INT32
    assert call(A=None) == -5
    assert call(lda=7) == -6
    assert call(B=None) == -7
    assert call(ldb=7) == -8
    assert call(Cm=None) == -10
    assert call(ldc=7) == -11
    assert call(num_moduli=1) == -12 and call(num_moduli=21) == -12
    assert call(scaling_mode=3) == -13 and call(scaling_mode=-1) == -13
    assert call(m=0) == 0 and call(n=0) == 0      # quick return before any device work
    assert "num_moduli" in B.ozaki2_status_string(-12)
    assert B.ozaki2_status_string(0) == "success"
    assert "workspace" in B.ozaki2_status_string(B.OZAKI2_ERR_WORKSPACE)


def test_workspace_size_formula(B):
    # N X + N Y (+ X for accurate mode) + small vectors: 3.2 GB at 8192^3, N = 16
    m = n = k = 8192
    w = B.ozaki2_workspace_bytes(m, n, k, 16, 2)
    assert 16 * (m * k + k * n) + 16 * m * n <= w <= 16 * (m * k + k * n) + 16 * m * n + (1 << 20)
    wa = B.ozaki2_workspace_bytes(m, n, k, 16, 0)
    assert wa - w >= m * k + k * n
    assert B.ozaki2_workspace_bytes(m, n, (1 << 22) + 1, 16, 2) == 0
    assert B.ozaki2_workspace_bytes(m, n, k, 21, 2) == 0
    assert B.ozaki2_host_scratch_bytes(4, 5, 6) >= 8 * (24 + 30 + 20)


@pytest.mark.parametrize("N", range(2, 21))
def test_library_constants_against_mpmath_and_theorem1(B, N, golden):
    c = B.ozaki2_get_constants(N)
    paper = [int(x) for x in golden("eq14_moduli.txt")["moduli"].split(",")]
    assert c["p"] == paper[:N]
    P = int(np.prod([int(x) for x in c["p"]], dtype=object))
    assert c["P"] == P
    for l in range(N):
        assert (P // c["p"][l] * c["q"][l]) % c["p"][l] == 1
        assert c["w"][l] == P // c["p"][l] * c["q"][l]
    assert sum(c["w"]) % P == 1
    mp.prec = 400
    l2 = log(mpf(P - 1), 2)

    def down(x):
        f = np.float32(float(x))
        return np.float32(np.nextafter(f, np.float32(-np.inf))) if mpf(float(f)) > x else f

    assert c["Pprop"] == down(l2 / 2 - mpf("0.5"))
    assert c["Pfast"] == down(l2 / 2 - mpf("1.5"))
    assert float(c["delta"]) == float.fromhex("0x1.000006p-1")


def test_blas_workspace_query_follows_the_layout(B):
    # a row-major BLAS-shaped call runs as the (n, m, k) problem; ozaki2_blas_workspace_bytes reports that orientation
    for m, n, k, N, mode in [(1, 300, 64, 14, 2), (300, 1, 64, 14, 2), (17, 4000, 129, 20, 0), (8192, 8192, 8192, 16, 2)]:
        assert B.ozaki2_blas_workspace_bytes("C", m, n, k, N, mode) == B.ozaki2_workspace_bytes(m, n, k, N, mode) > 0
        assert B.ozaki2_blas_workspace_bytes("r", m, n, k, N, mode) == B.ozaki2_workspace_bytes(n, m, k, N, mode) > 0
    assert B.ozaki2_blas_workspace_bytes("X", 8, 8, 8, 14, 2) == 0
    assert B.ozaki2_workspace_bytes(1, 300, 64, 14, 2) != B.ozaki2_workspace_bytes(300, 1, 64, 14, 2)
