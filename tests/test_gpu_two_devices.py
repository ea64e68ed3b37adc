"""Two GPUs used from one process (-m gpu; skipped on a one-GPU box).

include/ozaki2.h promises that calls on different devices are independent: each device has its own constant tables,
kernel attributes (the > 48 KB shared-memory opt-in of the CRT and GEMM kernels is a per-device setting) and workspace.
"""
import numpy as np
import pytest

import workloads as W
from oracle import ozaki2_oracle as O

pytestmark = pytest.mark.gpu


def test_dgemm_on_two_devices_from_one_process():
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    import paper_2606_29129_b200 as B
    B.lib()
    m, n, k, N = 300, 260, 700, 16
    A, Bm = W.eq15_matrices(m, n, k, 1.0, 5150)
    want = {mode: O.dgemm(A, Bm, N, mode) for mode in (2, 0)}
    for rounds in range(2):                           # the second round finds both devices already set up
        for dev in (1, 0):                            # the device that is NOT the process's first one goes first
            with torch.cuda.device(dev):
                Ad = torch.from_numpy(np.ascontiguousarray(A.T)).cuda(dev)
                Bd = torch.from_numpy(np.ascontiguousarray(Bm.T)).cuda(dev)
                for mode in (2, 0):
                    Cd = B.dgemm(Ad, Bd, N, mode)
                    torch.cuda.synchronize(dev)
                    assert np.array_equal(B.device_to_colmajor(Cd), want[mode]), (dev, mode)
                e = torch.empty((m,), dtype=torch.int32, device=f"cuda:{dev}")
                assert B.ozaki2_row_exponents_noalloc(m, k, Ad, m, N, 2, e) == 0
                torch.cuda.synchronize(dev)
                assert np.array_equal(e.cpu().numpy(), O.stages(A, Bm, N, 2)["e"])
