"""Thin Python binding of libozaki2.so (include/ozaki2.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch appears only as the owner of
device memory and streams.  There is no CPU fallback: a missing library raises at import of the
first call, a non-B200 device returns OZAKI2_ERR_DEVICE from the library.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libozaki2.so")

OZAKI2_MODE_ACCURATE, OZAKI2_MODE_FAST, OZAKI2_MODE_PROP = 0, 1, 2
OZAKI2_ERR_WORKSPACE, OZAKI2_ERR_DEVICE = -100, -101
OZAKI2_NOALLOC_MAX_ROWS, OZAKI2_ERR_NOALLOC_LIMIT = 65536, -102
OZAKI2_K_BLOCK, OZAKI2_MAX_K, OZAKI2_MAX_K_ACCURATE = 1 << 17, 1 << 22, 1 << 18

_lib = None


class Ozaki2Error(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status}: {ozaki2_status_string(status)}")


class ozaki2_stage_outputs(C.Structure):
    _fields_ = [("e", C.c_void_p), ("f", C.c_void_p), ("rowmax", C.c_void_p), ("colmax", C.c_void_p),
                ("resA", C.c_void_p), ("resB", C.c_void_p), ("U", C.c_void_p), ("Cpp", C.c_void_p),
                ("stage_ms", C.POINTER(C.c_float)), ("stage_events", C.POINTER(C.c_void_p))]


def lib() -> C.CDLL:
    """Load libozaki2.so; raises if it has not been built (python paper_2606_29129_b200/build.py)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} is missing: build it with `python paper_2606_29129_b200/build.py` "
                                    "(there is no fallback path)")
        L = C.CDLL(LIB_PATH)
        i64, dbl, vp, ci = C.c_int64, C.c_double, C.c_void_p, C.c_int
        gemm_args = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, ci, ci, vp]
        L.ozaki2_dgemm.argtypes = gemm_args
        L.ozaki2_dgemm.restype = ci
        L.ozaki2_dgemm_stages.argtypes = gemm_args + [C.POINTER(ozaki2_stage_outputs)]
        L.ozaki2_dgemm_stages.restype = ci
        L.ozaki2_dgemm_t.argtypes = [ci, ci] + gemm_args
        L.ozaki2_dgemm_t.restype = ci
        sgemm_args = [i64, i64, i64, C.c_float, vp, i64, vp, i64, C.c_float, vp, i64, ci, ci, vp]
        L.ozaki2_sgemm.argtypes = sgemm_args
        L.ozaki2_dgemm_ws.argtypes = gemm_args[:-1] + [vp, C.c_size_t, vp]
        L.ozaki2_dgemm_ws.restype = ci
        L.ozaki2_sgemm_ws.argtypes = sgemm_args[:-1] + [vp, C.c_size_t, vp]
        L.ozaki2_sgemm_ws.restype = ci
        L.ozaki2_sgemm.restype = ci
        L.ozaki2_sgemm_stages.argtypes = sgemm_args + [C.POINTER(ozaki2_stage_outputs)]
        L.ozaki2_sgemm_stages.restype = ci
        L.ozaki2_dgemm_host.argtypes = [i64, i64, i64, dbl, vp, i64, vp, i64, dbl, vp, i64, ci, ci, vp, C.c_size_t, vp]
        L.ozaki2_dgemm_host.restype = ci
        L.ozaki2_sgemm_host.argtypes = [i64, i64, i64, C.c_float, vp, i64, vp, i64, C.c_float, vp, i64, ci, ci, vp,
                                        C.c_size_t, vp]
        L.ozaki2_sgemm_host.restype = ci
        L.ozaki2_sgemm_t.argtypes = [ci, ci] + sgemm_args
        L.ozaki2_sgemm_t.restype = ci
        L.ozaki2_dgemm_blas.argtypes = [ci, ci, ci] + gemm_args
        L.ozaki2_dgemm_blas.restype = ci
        L.ozaki2_sgemm_blas.argtypes = [ci, ci, ci] + sgemm_args
        L.ozaki2_sgemm_blas.restype = ci
        L.ozaki2_zgemm.argtypes = [i64, i64, i64, dbl, dbl, vp, i64, vp, i64, dbl, dbl, vp, i64, ci, ci, vp]
        L.ozaki2_zgemm.restype = ci
        L.ozaki2_zgemm_workspace_bytes.argtypes = [i64, i64, i64, ci, ci]
        L.ozaki2_zgemm_workspace_bytes.restype = C.c_size_t
        L.ozaki2_cgemm.argtypes = [i64, i64, i64, C.c_float, C.c_float, vp, i64, vp, i64, C.c_float, C.c_float, vp, i64, ci, ci, vp]
        L.ozaki2_cgemm.restype = ci
        L.ozaki2_cgemm_workspace_bytes.argtypes = [i64, i64, i64, ci, ci]
        L.ozaki2_cgemm_workspace_bytes.restype = C.c_size_t
        L.ozaki2_debug_crt.argtypes = [ci, i64, i64, vp, vp, vp, dbl, dbl, vp, i64, vp, ci, vp]
        L.ozaki2_debug_crt.restype = ci
        L.ozaki2_workspace_bytes.argtypes = [i64, i64, i64, ci, ci]
        L.ozaki2_workspace_bytes.restype = C.c_size_t
        L.ozaki2_blas_workspace_bytes.argtypes = [ci, i64, i64, i64, ci, ci]
        L.ozaki2_blas_workspace_bytes.restype = C.c_size_t
        L.ozaki2_host_scratch_bytes.argtypes = [i64, i64, i64]
        L.ozaki2_host_scratch_bytes.restype = C.c_size_t
        L.ozaki2_set_workspace.argtypes = [vp, C.c_size_t]
        L.ozaki2_set_workspace.restype = ci
        L.ozaki2_status_string.argtypes = [ci]
        L.ozaki2_status_string.restype = C.c_char_p
        L.ozaki2_get_constants.argtypes = [ci, vp, vp, vp, vp, C.POINTER(C.c_float), C.POINTER(C.c_float),
                                           C.POINTER(C.c_float)]
        L.ozaki2_get_constants.restype = ci
        L.ozaki2_debug_log2f.argtypes = [vp, vp, i64, vp]
        L.ozaki2_debug_log2f.restype = ci
        L.ozaki2_debug_mod_p.argtypes = [ci, vp, vp, i64, vp]
        L.ozaki2_debug_mod_p.restype = ci
        L.ozaki2_debug_residue_gemm.argtypes = [ci, i64, i64, i64, vp, vp, vp, ci, vp]
        L.ozaki2_debug_residue_gemm.restype = ci
        L.ozaki2_row_exponents_noalloc.argtypes = [i64, i64, vp, i64, ci, ci, vp, vp]
        L.ozaki2_row_exponents_noalloc.restype = ci
        L.ozaki2_version.restype = C.c_char_p
        L.ozaki2_kernel_launches.argtypes = []
        L.ozaki2_kernel_launches.restype = C.c_uint64
        _lib = L
    return _lib


def _ptr(x):
    """torch tensor / numpy array / int / None -> raw address."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()          # torch.Tensor


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def ozaki2_status_string(status: int) -> str:
    return lib().ozaki2_status_string(int(status)).decode()


def ozaki2_version() -> str:
    return lib().ozaki2_version().decode()


def ozaki2_kernel_launches() -> int:
    return int(lib().ozaki2_kernel_launches())


def ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode) -> int:
    return int(lib().ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode))


def ozaki2_host_scratch_bytes(m, n, k) -> int:
    return int(lib().ozaki2_host_scratch_bytes(m, n, k))


def ozaki2_set_workspace(device_ptr, nbytes) -> int:
    return int(lib().ozaki2_set_workspace(_ptr(device_ptr), nbytes))


def ozaki2_dgemm(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    """Raw call: returns the library's status (0 = success).  A, B, Cm: device tensors or addresses."""
    return int(lib().ozaki2_dgemm(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli,
                                  scaling_mode, _stream(stream)))


def ozaki2_dgemm_ws(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, workspace, workspace_bytes,
                    stream=None) -> int:
    """ozaki2_dgemm with the workspace of this call passed in (device tensor or address): independent of other calls."""
    return int(lib().ozaki2_dgemm_ws(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli, scaling_mode,
                                     _ptr(workspace), workspace_bytes, _stream(stream)))


def ozaki2_sgemm_ws(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, workspace, workspace_bytes,
                    stream=None) -> int:
    return int(lib().ozaki2_sgemm_ws(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli, scaling_mode,
                                     _ptr(workspace), workspace_bytes, _stream(stream)))


def ozaki2_dgemm_stages(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None,
                        out: ozaki2_stage_outputs | None = None) -> int:
    return int(lib().ozaki2_dgemm_stages(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli,
                                         scaling_mode, _stream(stream), C.byref(out) if out is not None else None))


def ozaki2_dgemm_t(transa, transb, m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    return int(lib().ozaki2_dgemm_t(transa, transb, m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc,
                                    num_moduli, scaling_mode, _stream(stream)))


def ozaki2_sgemm(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    """SGEMM variant: A, B, Cm are FP32 device tensors or addresses."""
    return int(lib().ozaki2_sgemm(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli,
                                  scaling_mode, _stream(stream)))


def ozaki2_sgemm_stages(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None,
                        out: ozaki2_stage_outputs | None = None) -> int:
    return int(lib().ozaki2_sgemm_stages(m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc, num_moduli,
                                         scaling_mode, _stream(stream), C.byref(out) if out is not None else None))


def ozaki2_dgemm_host(m, n, k, alpha, A_host, lda, B_host, ldb, beta, C_host, ldc, num_moduli, scaling_mode,
                      device_scratch, scratch_bytes, stream=None) -> int:
    return int(lib().ozaki2_dgemm_host(m, n, k, alpha, _ptr(A_host), lda, _ptr(B_host), ldb, beta, _ptr(C_host), ldc,
                                       num_moduli, scaling_mode, _ptr(device_scratch), scratch_bytes, _stream(stream)))


def ozaki2_sgemm_host(m, n, k, alpha, A_host, lda, B_host, ldb, beta, C_host, ldc, num_moduli, scaling_mode,
                      device_scratch, scratch_bytes, stream=None) -> int:
    return int(lib().ozaki2_sgemm_host(m, n, k, alpha, _ptr(A_host), lda, _ptr(B_host), ldb, beta, _ptr(C_host), ldc,
                                       num_moduli, scaling_mode, _ptr(device_scratch), scratch_bytes, _stream(stream)))


def ozaki2_sgemm_t(transa, transb, m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    return int(lib().ozaki2_sgemm_t(transa, transb, m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb, beta, _ptr(Cm), ldc,
                                    num_moduli, scaling_mode, _stream(stream)))


def _flag(c):
    """'N' / 'T' / 'C' / 'R' (str or bytes) or a CBLAS enum -> int"""
    return c if isinstance(c, int) else ord(c)


def ozaki2_dgemm_blas(layout, transa, transb, m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode,
                      stream=None) -> int:
    return int(lib().ozaki2_dgemm_blas(_flag(layout), _flag(transa), _flag(transb), m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb,
                                       beta, _ptr(Cm), ldc, num_moduli, scaling_mode, _stream(stream)))


def ozaki2_sgemm_blas(layout, transa, transb, m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode,
                      stream=None) -> int:
    return int(lib().ozaki2_sgemm_blas(_flag(layout), _flag(transa), _flag(transb), m, n, k, alpha, _ptr(A), lda, _ptr(B), ldb,
                                       beta, _ptr(Cm), ldc, num_moduli, scaling_mode, _stream(stream)))


def ozaki2_blas_workspace_bytes(layout, m, n, k, num_moduli, scaling_mode) -> int:
    return int(lib().ozaki2_blas_workspace_bytes(_flag(layout), m, n, k, num_moduli, scaling_mode))


def ozaki2_zgemm_workspace_bytes(m, n, k, num_moduli, scaling_mode) -> int:
    return int(lib().ozaki2_zgemm_workspace_bytes(m, n, k, num_moduli, scaling_mode))


def ozaki2_zgemm(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    """Complex variant: A, B, Cm are complex128 device tensors (column-major) or addresses; alpha, beta complex."""
    alpha, beta = complex(alpha), complex(beta)
    return int(lib().ozaki2_zgemm(m, n, k, alpha.real, alpha.imag, _ptr(A), lda, _ptr(B), ldb, beta.real, beta.imag, _ptr(Cm), ldc,
                                  num_moduli, scaling_mode, _stream(stream)))


def ozaki2_cgemm_workspace_bytes(m, n, k, num_moduli, scaling_mode) -> int:
    return int(lib().ozaki2_cgemm_workspace_bytes(m, n, k, num_moduli, scaling_mode))


def ozaki2_cgemm(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream=None) -> int:
    """Single-precision complex variant: A, B, Cm are complex64 device tensors (column-major) or addresses."""
    alpha, beta = complex(alpha), complex(beta)
    return int(lib().ozaki2_cgemm(m, n, k, alpha.real, alpha.imag, _ptr(A), lda, _ptr(B), ldb, beta.real, beta.imag, _ptr(Cm), ldc,
                                  num_moduli, scaling_mode, _stream(stream)))


def ensure_zgemm_workspace(m, n, k, num_moduli, scaling_mode):
    """Allocate (grow-only) and register a workspace large enough for ozaki2_zgemm (and ozaki2_cgemm) on the current device."""
    import torch
    need = ozaki2_zgemm_workspace_bytes(m, n, k, num_moduli, scaling_mode)
    dev = torch.cuda.current_device()
    cur = _ws_tensor.get(dev)
    if cur is None or cur.numel() < need:
        _ws_tensor[dev] = None
        cur = torch.empty(max(need, 256), dtype=torch.uint8, device=f"cuda:{dev}")
        _ws_tensor[dev] = cur
    rc = ozaki2_set_workspace(cur, cur.numel())
    if rc:
        raise Ozaki2Error(rc, "ozaki2_set_workspace")
    return cur


def ozaki2_debug_crt(num_moduli, m, n, U, e, f, alpha, beta, Cm, ldc, Cpp=None, is_f32=False, stream=None) -> int:
    return int(lib().ozaki2_debug_crt(num_moduli, m, n, _ptr(U), _ptr(e), _ptr(f), alpha, beta, _ptr(Cm), ldc, _ptr(Cpp),
                                      1 if is_f32 else 0, _stream(stream)))


def ozaki2_row_exponents_noalloc(m, k, A, lda, num_moduli, scaling_mode, e, stream=None) -> int:
    """e[i] = log2 mu_i for the m rows of the column-major device matrix A (fast / revised fast mode), computed with the
    library's built-in scratch array instead of a workspace: the call for code that is not in a position to allocate
    device memory (see include/ozaki2.h).  A, e: device tensors or addresses; at most OZAKI2_NOALLOC_MAX_ROWS rows;
    calls on one device share the scratch and must not overlap on the GPU.  Returns the library's status."""
    return int(lib().ozaki2_row_exponents_noalloc(m, k, _ptr(A), lda, num_moduli, scaling_mode, _ptr(e), _stream(stream)))


def ozaki2_get_constants(num_moduli: int) -> dict:
    N = num_moduli
    p = np.zeros(20, np.int32)
    q = np.zeros(20, np.int32)
    P = np.zeros(4, np.uint64)
    w = np.zeros((20, 4), np.uint64)
    a, b, d = C.c_float(), C.c_float(), C.c_float()
    rc = lib().ozaki2_get_constants(N, p.ctypes.data, q.ctypes.data, P.ctypes.data, w.ctypes.data, C.byref(a),
                                    C.byref(b), C.byref(d))
    if rc:
        raise Ozaki2Error(rc, "ozaki2_get_constants")

    def to_int(words):
        return sum(int(words[t]) << (64 * t) for t in range(4))

    return dict(N=N, p=[int(x) for x in p[:N]], q=[int(x) for x in q[:N]], P=to_int(P),
                w=[to_int(w[l]) for l in range(N)], Pprop=np.float32(a.value), Pfast=np.float32(b.value),
                delta=np.float32(d.value))


def ozaki2_debug_log2f(x, y, count, stream=None) -> int:
    return int(lib().ozaki2_debug_log2f(_ptr(x), _ptr(y), count, _stream(stream)))


def ozaki2_debug_mod_p(modulus_index, inp, out, count, stream=None) -> int:
    return int(lib().ozaki2_debug_mod_p(modulus_index, _ptr(inp), _ptr(out), count, _stream(stream)))


def ozaki2_debug_residue_gemm(num_moduli, m, n, k, resA, resB, U, use_tensor_cores=1, stream=None) -> int:
    return int(lib().ozaki2_debug_residue_gemm(num_moduli, m, n, k, _ptr(resA), _ptr(resB), _ptr(U),
                                               use_tensor_cores, _stream(stream)))


# ------------------------------------------------------------------------------------------------
# conveniences on top of the raw calls (device memory through torch; still no arithmetic here)
# ------------------------------------------------------------------------------------------------
_ws_tensor = {}


def ensure_workspace(m, n, k, num_moduli, scaling_mode):
    """Allocate (grow-only) and register the workspace of the current device."""
    import torch
    need = ozaki2_workspace_bytes(m, n, k, num_moduli, scaling_mode)
    dev = torch.cuda.current_device()
    cur = _ws_tensor.get(dev)
    if cur is None or cur.numel() < need:
        _ws_tensor[dev] = None
        cur = torch.empty(max(need, 256), dtype=torch.uint8, device=f"cuda:{dev}")
        _ws_tensor[dev] = cur
    rc = ozaki2_set_workspace(cur, cur.numel())
    if rc:
        raise Ozaki2Error(rc, "ozaki2_set_workspace")
    return cur


def colmajor_to_device(a: np.ndarray, dtype=np.float64):
    """numpy (rows, cols) matrix -> device tensor of shape (cols, rows) whose memory is the column-major matrix."""
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=dtype).T)).cuda()


def device_to_colmajor(t) -> np.ndarray:
    """inverse of colmajor_to_device: returns a Fortran-ordered (rows, cols) numpy array."""
    return np.asfortranarray(t.cpu().numpy().T)


def dgemm(A_dev, B_dev, num_moduli, scaling_mode=OZAKI2_MODE_PROP, alpha=1.0, beta=0.0, C_dev=None, stream=None):
    """C = alpha A B + beta C on column-major device matrices (tensors of shape (cols, rows), see above)."""
    import torch
    k, m = A_dev.shape
    n, k2 = B_dev.shape
    assert k == k2 and A_dev.dtype == torch.float64 and B_dev.dtype == torch.float64
    if C_dev is None:
        C_dev = torch.empty((n, m), dtype=torch.float64, device=A_dev.device)
    ensure_workspace(m, n, k, num_moduli, scaling_mode)
    rc = ozaki2_dgemm(m, n, k, alpha, A_dev, max(1, m), B_dev, max(1, k), beta, C_dev, max(1, m), num_moduli,
                      scaling_mode, stream)
    if rc:
        raise Ozaki2Error(rc, "ozaki2_dgemm")
    return C_dev


def dgemm_with_stage_events(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, events, stream=None,
                            f32=False) -> int:
    """ozaki2_dgemm_stages with nothing but `stage_events`: the same kernels as ozaki2_dgemm, plus five
    cudaEventRecord calls.  `events`: five torch.cuda.Event(enable_timing=True) that have been recorded once
    (torch creates the CUDA event lazily).  No synchronisation."""
    out = ozaki2_stage_outputs()
    arr = (C.c_void_p * 5)(*[ev.cuda_event for ev in events])
    out.stage_events = C.cast(arr, C.POINTER(C.c_void_p))
    call = ozaki2_sgemm_stages if f32 else ozaki2_dgemm_stages
    return call(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, num_moduli, scaling_mode, stream, out)


def dgemm_stages(A_dev, B_dev, num_moduli, scaling_mode, alpha=1.0, beta=0.0, C_dev=None, want=("e", "f", "resA", "resB", "U", "Cpp"),
                 timing=False, stream=None) -> dict:
    """Run the path and return the requested intermediate results (device tensors, canonical layouts)."""
    import torch
    k, m = A_dev.shape
    n, _ = B_dev.shape
    N = num_moduli
    dev = A_dev.device
    f32 = A_dev.dtype == torch.float32
    if C_dev is None:
        C_dev = torch.empty((n, m), dtype=A_dev.dtype, device=dev)
    ensure_workspace(m, n, k, N, scaling_mode)
    bufs = {}
    shapes = dict(e=((m,), torch.int32), f=((n,), torch.int32), rowmax=((m,), torch.int32), colmax=((n,), torch.int32),
                  resA=((N, m, k), torch.int8), resB=((N, n, k), torch.int8), U=((N, n, m), torch.uint8),
                  Cpp=((n, m, 4), torch.int64))
    out = ozaki2_stage_outputs()
    for name in want:
        shp, dt = shapes[name]
        bufs[name] = torch.zeros(shp, dtype=dt, device=dev)
        setattr(out, name, bufs[name].data_ptr())
    ms = (C.c_float * 5)()
    if timing:
        out.stage_ms = C.cast(ms, C.POINTER(C.c_float))
    call = ozaki2_sgemm_stages if f32 else ozaki2_dgemm_stages
    rc = call(m, n, k, alpha, A_dev, max(1, m), B_dev, max(1, k), beta, C_dev, max(1, m), N, scaling_mode, stream, out)
    if rc:
        raise Ozaki2Error(rc, "ozaki2_sgemm_stages" if f32 else "ozaki2_dgemm_stages")
    bufs["C"] = C_dev
    if timing:
        bufs["stage_ms"] = [float(x) for x in ms]
    return bufs
