"""Thin Python binding of libmp_b200.so (include/mp_b200.h).  Argument marshalling only: every step
of the Matching Pursuit path runs in the library's CUDA kernels.  PyTorch supplies device memory and
streams.  There is no CPU fallback: a missing library or a failed call raises.

Function names and argument order follow the C header; see include/mp_b200.h for the contract
(citations into PAPER.md, layouts, ownership, error behaviour).
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))


class MPError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"mp_b200 status {status} ({_STATUS.get(status, '?')}): {message}")
        self.status = status


_STATUS = {0: "MP_OK", 1: "MP_ERR_INVALID_ARG", 2: "MP_ERR_CUDA", 3: "MP_ERR_UNSUPPORTED", 4: "MP_ERR_WORKSPACE"}
MP_OK, MP_ERR_INVALID_ARG, MP_ERR_CUDA, MP_ERR_UNSUPPORTED, MP_ERR_WORKSPACE = range(5)


def _load():
    """build() is a no-op when the library is newer than every source it depends on, so a stale libmp_b200.so (git-ignored, but
    shipped with the tree) is never loaded silently after an edit of csrc/."""
    path = _build.LIB
    try:
        _build.build()
    except Exception as e:  # loud: no fallback implementation exists
        if not os.path.exists(path):
            raise ImportError(f"libmp_b200.so is missing and could not be built with nvcc: {e}") from e
        import warnings
        warnings.warn(f"libmp_b200.so could not be rebuilt ({e}); loading the existing library, which may be older than csrc/")
    return C.CDLL(path)


lib = _load()
_vp, _i, _i64, _f, _sz = C.c_void_p, C.c_int, C.c_int64, C.c_float, C.c_size_t
lib.mp_workspace_bytes.restype = _sz
lib.mp_workspace_bytes.argtypes = [_i, _i, _i]
lib.mp_normalize_columns.restype = _i
lib.mp_normalize_columns.argtypes = [_vp, _i, _i, _i64, _vp, _vp]
lib.mp_recover.restype = _i
lib.mp_recover.argtypes = [_vp, _i, _i, _i64, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
lib.mp_recover_noalloc.restype = _i
lib.mp_recover_noalloc.argtypes = [_vp, _i, _i, _i64, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp, _vp]
lib.mp_recover_batched.restype = _i
lib.mp_recover_batched.argtypes = [_vp, _i, _i, _i64, _vp, _i64, _i, _f, _i, _vp, _vp, _vp, _vp, _sz, _vp]
lib.mp_recover_batched_traced.restype = _i
lib.mp_recover_batched_traced.argtypes = [_vp, _i, _i, _i64, _vp, _i64, _i, _f, _i, _vp, _vp, _vp, _vp, _vp, _i64, _vp, _sz, _vp]
lib.mp_correlate_batched_workspace_bytes.restype = _sz
lib.mp_correlate_batched_workspace_bytes.argtypes = [_i, _i, _i]
lib.mp_correlate_batched.restype = _i
lib.mp_correlate_batched.argtypes = [_vp, _i, _i, _i64, _vp, _i64, _i, _vp, _vp, _sz, _vp]
lib.mp_encode_sparse.restype = _i
lib.mp_encode_sparse.argtypes = [_vp, _i, _i, _i64, _vp, _vp, _i, _vp, _vp]
lib.mp_reconstruction_error.restype = _i
lib.mp_reconstruction_error.argtypes = [_vp, _vp, _i, _vp, _vp]
lib.mp_workspace_bytes_f64.restype = _sz
lib.mp_workspace_bytes_f64.argtypes = [_i, _i]
lib.mp_normalize_columns_f64.restype = _i
lib.mp_normalize_columns_f64.argtypes = [_vp, _i, _i, _i64, _vp, _vp]
lib.mp_recover_f64.restype = _i
lib.mp_recover_f64.argtypes = [_vp, _i, _i, _i64, _vp, C.c_double, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
lib.mp_workspace_bytes_omp.restype = _sz
lib.mp_workspace_bytes_omp.argtypes = [_i, _i, _i]
lib.mp_recover_omp.restype = _i
lib.mp_recover_omp.argtypes = [_vp, _i, _i, _i64, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
lib.mp_pack_signs.restype = _i
lib.mp_pack_signs.argtypes = [_vp, _i, _i, _i64, _vp, _i64, _vp, _vp, _vp]
lib.mp_recover_signs.restype = _i
lib.mp_recover_signs.argtypes = [_vp, _i, _i, _i64, _f, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
lib.mp_transpose_rowmajor.restype = _i
lib.mp_transpose_rowmajor.argtypes = [_vp, _i, _i, _i64, _vp, _i64, _vp]
lib.mp_workspace_bytes_many.restype = _sz
lib.mp_workspace_bytes_many.argtypes = [_i, _i, _i]
lib.mp_recover_many.restype = _i
lib.mp_recover_many.argtypes = [_vp, _i, _i, _i64, _i64, _vp, _i64, _i, _f, _i, _vp, _vp, _vp, _vp, _vp, _i64, _vp, _sz, _vp]
lib.mp_workspace_bytes_signs_many.restype = _sz
lib.mp_workspace_bytes_signs_many.argtypes = [_i, _i, _i]
lib.mp_recover_signs_many.restype = _i
lib.mp_recover_signs_many.argtypes = [_vp, _i, _i, _i64, _i64, _f, _vp, _i64, _i, _f, _i, _vp, _vp, _vp, _vp, _vp, _i64, _vp, _sz, _vp]
lib.mp_last_error.restype = C.c_char_p
lib.mp_last_error.argtypes = []
lib.mp_set_int.restype = _i
lib.mp_set_int.argtypes = [C.c_char_p, _i64]
lib.mp_get_int.restype = _i
lib.mp_get_int.argtypes = [C.c_char_p, C.POINTER(_i64)]
lib.mp_probe_read.restype = _i
lib.mp_probe_read.argtypes = [_vp, _sz, _i, _vp, C.POINTER(C.c_ulonglong), _vp]
lib.mp_launch_count.restype = _i64
lib.mp_launch_count.argtypes = []
lib.mp_recover_host.restype = _i
lib.mp_recover_host.argtypes = [_vp, _i, _i, _i64, _i, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp]
lib.mp_recover_batched_host.restype = _i
lib.mp_recover_batched_host.argtypes = [_vp, _i, _i, _i64, _i, _vp, _i64, _i, _f, _i, _vp, _vp, _vp]
lib.mp_dictionary_create.restype = _i
lib.mp_dictionary_create.argtypes = [_vp, _i, _i, _i, _i64, _i, C.POINTER(_vp)]
lib.mp_dictionary_destroy.restype = _i
lib.mp_dictionary_destroy.argtypes = [_vp]
lib.mp_dictionary_info.restype = _i
lib.mp_dictionary_info.argtypes = [_vp, C.POINTER(_i), C.POINTER(_i), C.POINTER(_i64), C.POINTER(_vp)]
lib.mp_recover_host_h.restype = _i
lib.mp_recover_host_h.argtypes = [_vp, _vp, _f, _i, _vp, _vp, _vp, _vp, _vp]
lib.mp_recover_batched_host_h.restype = _i
lib.mp_recover_batched_host_h.argtypes = [_vp, _vp, _i64, _i, _f, _i, _vp, _vp, _vp, _vp, _vp, _i64]


def _check(status: int):
    if status != 0:
        raise MPError(status, lib.mp_last_error().decode())


def mp_last_error() -> str:
    return lib.mp_last_error().decode()


def mp_set_int(name: str, value: int) -> None:
    _check(lib.mp_set_int(name.encode(), int(value)))


def mp_get_int(name: str) -> int:
    v = _i64(0)
    _check(lib.mp_get_int(name.encode(), C.byref(v)))
    return v.value


def mp_launch_count() -> int:
    return lib.mp_launch_count()


def mp_probe_read(buf: torch.Tensor, passes: int, *, sink: torch.Tensor | None = None, stream=None) -> int:
    """The read-only streaming diagnostic (include/mp_b200.h): enqueues `passes` reads of the device tensor `buf` and returns the
    number of bytes the launch reads; the caller times it with CUDA events."""
    if not (buf.is_cuda and buf.is_contiguous()):
        raise TypeError("buf must be a contiguous CUDA tensor")
    sink = torch.zeros(1, dtype=torch.float32, device=buf.device) if sink is None else sink
    n = C.c_ulonglong(0)
    with torch.cuda.device(buf.device):
        _check(lib.mp_probe_read(buf.data_ptr(), buf.numel() * buf.element_size(), int(passes), _dev(sink, torch.float32, "sink"),
                                 C.byref(n), _stream_ptr(stream)))
    buf._mp_sink = sink                 # keep the sink alive until the stream has run the kernel
    return n.value


def mp_workspace_bytes(N: int, M: int, B: int = 1) -> int:
    return lib.mp_workspace_bytes(N, M, B)


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


def _dict_args(psi_t: torch.Tensor):
    if not (psi_t.is_cuda and psi_t.dtype == torch.float32 and psi_t.dim() == 2 and (psi_t.shape[1] == 1 or psi_t.stride(1) == 1)):
        raise TypeError("psi_t must be a CUDA float32 [M, N] tensor with unit stride along N (atom-major)")
    M, N = psi_t.shape
    ld = psi_t.stride(0) if M > 1 else max(psi_t.stride(0), N)
    return psi_t.data_ptr(), N, M, ld


def _dev(t: torch.Tensor, dtype, what: str):
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous CUDA {dtype} tensor")
    return t.data_ptr()


def _workspace(N, M, B, workspace, device):
    need = mp_workspace_bytes(N, M, B)
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=device)
    base = workspace.data_ptr()
    off = (-base) % 256
    return workspace, base + off, workspace.numel() - off


def mp_normalize_columns(psi_t: torch.Tensor, norms_out: torch.Tensor | None = None, stream=None) -> None:
    """Eq. 4, in place on the device tensor psi_t[M, N]."""
    p, N, M, ld = _dict_args(psi_t)
    n = _dev(norms_out, torch.float32, "norms_out") if norms_out is not None else None
    with torch.cuda.device(psi_t.device):
        _check(lib.mp_normalize_columns(p, N, M, ld, n, _stream_ptr(stream)))


def mp_transpose_rowmajor(psi: torch.Tensor, psi_t: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """The paper's row-major Psi[N, M] (A2 P:360) -> the atom-major psi_t[M, N] the solvers take (row stride padded to 4)."""
    if not (psi.is_cuda and psi.dtype == torch.float32 and psi.dim() == 2 and (psi.shape[1] == 1 or psi.stride(1) == 1)):
        raise TypeError("psi must be a CUDA float32 [N, M] tensor with unit stride along M (row-major Psi)")
    N, M = psi.shape
    ldr = psi.stride(0) if N > 1 else max(psi.stride(0), M)
    if psi_t is None:
        ld = (N + 3) // 4 * 4
        psi_t = torch.zeros((M, ld), dtype=torch.float32, device=psi.device)[:, :N]
    p, N2, M2, ld = _dict_args(psi_t)
    if (N2, M2) != (N, M):
        raise ValueError("psi_t must be [M, N]")
    with torch.cuda.device(psi.device):
        _check(lib.mp_transpose_rowmajor(psi.data_ptr(), N, M, ldr, p, ld, _stream_ptr(stream)))
    return psi_t


@dataclasses.dataclass
class Recovered:
    x: torch.Tensor                      # [M] (or [B, M]) float32, device
    r: torch.Tensor                      # [N] (or [B, N]) float32, device
    n_iter: torch.Tensor                 # [1] (or [B]) int32, device
    idx_trace: torch.Tensor | None = None
    c_trace: torch.Tensor | None = None
    workspace: torch.Tensor | None = None


def mp_recover(psi_t: torch.Tensor, y: torch.Tensor, eps: float, max_iter: int, *, x=None, r=None, n_iter=None,
               idx_trace=None, c_trace=None, trace: bool = False, workspace=None, stream=None) -> Recovered:
    """Eq. 8-12 for one signal; asynchronous on the stream, outputs are device tensors."""
    p, N, M, ld = _dict_args(psi_t)
    dev = psi_t.device
    if y.numel() != N:
        raise ValueError("y must have N elements")
    x = torch.empty(M, dtype=torch.float32, device=dev) if x is None else x
    r = torch.empty(N, dtype=torch.float32, device=dev) if r is None else r
    n_iter = torch.empty(1, dtype=torch.int32, device=dev) if n_iter is None else n_iter
    if trace and idx_trace is None:
        idx_trace = torch.empty(max(max_iter, 1), dtype=torch.int32, device=dev)
    if trace and c_trace is None:
        c_trace = torch.empty(max(max_iter, 1), dtype=torch.float32, device=dev)
    workspace, wp, wb = _workspace(N, M, 1, workspace, dev)
    with torch.cuda.device(dev):
        _check(lib.mp_recover(p, N, M, ld, _dev(y, torch.float32, "y"), float(eps), int(max_iter),
                              _dev(x, torch.float32, "x"), _dev(r, torch.float32, "r"), _dev(n_iter, torch.int32, "n_iter"),
                              _dev(idx_trace, torch.int32, "idx_trace") if idx_trace is not None else None,
                              _dev(c_trace, torch.float32, "c_trace") if c_trace is not None else None,
                              wp, wb, _stream_ptr(stream)))
    return Recovered(x, r, n_iter, idx_trace, c_trace, workspace)


MP_NOALLOC_MAX_M = 65536


def mp_recover_noalloc(psi_t: torch.Tensor, y: torch.Tensor, eps: float, max_iter: int, *, x=None, r=None, n_iter=None,
                       idx_trace=None, c_trace=None, trace: bool = False, stream=None) -> Recovered:
    """mp_recover without a workspace, for callers that cannot allocate device memory (a plug-in inside a process whose own
    pool owns the GPU, a loop that must not stall on an allocation): the C call uses a fixed scratch array inside the library
    and allocates nothing.  M <= MP_NOALLOC_MAX_M; calls that overlap on the GPU race on that array (include/mp_b200.h).
    Pass x, r, n_iter (and the traces) to keep this wrapper from allocating too: any output left None is a fresh torch tensor."""
    p, N, M, ld = _dict_args(psi_t)
    dev = psi_t.device
    if y.numel() != N:
        raise ValueError("y must have N elements")
    x = torch.empty(M, dtype=torch.float32, device=dev) if x is None else x
    r = torch.empty(N, dtype=torch.float32, device=dev) if r is None else r
    n_iter = torch.empty(1, dtype=torch.int32, device=dev) if n_iter is None else n_iter
    if trace and idx_trace is None:
        idx_trace = torch.empty(max(max_iter, 1), dtype=torch.int32, device=dev)
    if trace and c_trace is None:
        c_trace = torch.empty(max(max_iter, 1), dtype=torch.float32, device=dev)
    with torch.cuda.device(dev):
        _check(lib.mp_recover_noalloc(p, N, M, ld, _dev(y, torch.float32, "y"), float(eps), int(max_iter),
                                      _dev(x, torch.float32, "x"), _dev(r, torch.float32, "r"), _dev(n_iter, torch.int32, "n_iter"),
                                      _dev(idx_trace, torch.int32, "idx_trace") if idx_trace is not None else None,
                                      _dev(c_trace, torch.float32, "c_trace") if c_trace is not None else None,
                                      _stream_ptr(stream)))
    return Recovered(x, r, n_iter, idx_trace, c_trace, None)


def mp_recover_batched(psi_t: torch.Tensor, Y: torch.Tensor, eps: float, max_iter: int, *, X=None, R=None, n_iter=None,
                       idx_trace=None, c_trace=None, trace: bool = False, workspace=None, stream=None) -> Recovered:
    """B signals sharing psi_t: Y[B, N] -> X[B, M], R[B, N], n_iter[B] (+ traces [B, max_iter] if asked)."""
    p, N, M, ld = _dict_args(psi_t)
    dev = psi_t.device
    if not (Y.is_cuda and Y.dtype == torch.float32 and Y.dim() == 2 and Y.shape[1] == N and (N == 1 or Y.stride(1) == 1)):
        raise TypeError("Y must be a CUDA float32 [B, N] tensor with unit stride along N")
    B = Y.shape[0]
    ldy = Y.stride(0) if B > 1 else max(Y.stride(0), N)
    X = torch.empty(B, M, dtype=torch.float32, device=dev) if X is None else X
    R = torch.empty(B, N, dtype=torch.float32, device=dev) if R is None else R
    n_iter = torch.empty(B, dtype=torch.int32, device=dev) if n_iter is None else n_iter
    if trace and idx_trace is None:
        idx_trace = torch.empty(B, max(max_iter, 1), dtype=torch.int32, device=dev)
    if trace and c_trace is None:
        c_trace = torch.empty(B, max(max_iter, 1), dtype=torch.float32, device=dev)
    ldt = max(max_iter, 1)
    for t_ in (idx_trace, c_trace):
        if t_ is not None and tuple(t_.shape) != (B, ldt):
            raise ValueError("traces must have shape [B, max(max_iter, 1)]")
    workspace, wp, wb = _workspace(N, M, B, workspace, dev)
    with torch.cuda.device(dev):
        _check(lib.mp_recover_batched_traced(
            p, N, M, ld, Y.data_ptr(), ldy, B, float(eps), int(max_iter),
            _dev(X, torch.float32, "X"), _dev(R, torch.float32, "R"), _dev(n_iter, torch.int32, "n_iter"),
            _dev(idx_trace, torch.int32, "idx_trace") if idx_trace is not None else None,
            _dev(c_trace, torch.float32, "c_trace") if c_trace is not None else None, ldt,
            wp, wb, _stream_ptr(stream)))
    return Recovered(X, R, n_iter, idx_trace, c_trace, workspace)


def mp_recover_many(psi_t: torch.Tensor, Y: torch.Tensor, eps: float, max_iter: int, *, trace: bool = False,
                    workspace=None, stream=None) -> Recovered:
    """P independent problems of one shape (the paper's Fig. 1 workload): psi_t[P, M, N] (or [M, N]: one shared
    dictionary), Y[P, N] -> X[P, M], R[P, N], n_iter[P] (+ traces [P, max_iter]); one thread-block cluster per problem."""
    if not (psi_t.is_cuda and psi_t.dtype == torch.float32 and psi_t.dim() in (2, 3) and (psi_t.shape[-1] == 1 or psi_t.stride(-1) == 1)):
        raise TypeError("psi_t must be a CUDA float32 [P, M, N] (or [M, N]) tensor with unit stride along N")
    M, N = psi_t.shape[-2:]
    dev = psi_t.device
    if not (Y.is_cuda and Y.dtype == torch.float32 and Y.dim() == 2 and Y.shape[1] == N and (N == 1 or Y.stride(1) == 1)):
        raise TypeError("Y must be a CUDA float32 [P, N] tensor with unit stride along N")
    P = Y.shape[0]
    ld = psi_t.stride(-2) if M > 1 else max(psi_t.stride(-2), N)
    if psi_t.dim() == 3:
        if psi_t.shape[0] != P:
            raise ValueError("psi_t[P, M, N] and Y[P, N] disagree on P")
        pstride = psi_t.stride(0) if P > 1 else max(psi_t.stride(0), M * ld)
    else:
        pstride = 0
    ldy = Y.stride(0) if P > 1 else max(Y.stride(0), N)
    X = torch.empty(P, M, dtype=torch.float32, device=dev)
    R = torch.empty(P, N, dtype=torch.float32, device=dev)
    n_iter = torch.empty(P, dtype=torch.int32, device=dev)
    ldt = max(max_iter, 1)
    idx_trace = torch.empty(P, ldt, dtype=torch.int32, device=dev) if trace else None
    c_trace = torch.empty(P, ldt, dtype=torch.float32, device=dev) if trace else None
    need = lib.mp_workspace_bytes_many(N, M, P)
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=dev)
    base = workspace.data_ptr()
    off = (-base) % 256
    with torch.cuda.device(dev):
        _check(lib.mp_recover_many(psi_t.data_ptr(), N, M, ld, pstride, Y.data_ptr(), ldy, P, float(eps), int(max_iter),
                                   X.data_ptr(), R.data_ptr(), n_iter.data_ptr(),
                                   idx_trace.data_ptr() if trace else None, c_trace.data_ptr() if trace else None, ldt,
                                   base + off, workspace.numel() - off, _stream_ptr(stream)))
    return Recovered(X, R, n_iter, idx_trace, c_trace, workspace)


def mp_correlate_batched(psi_t: torch.Tensor, Y: torch.Tensor, *, C_out=None, stream=None) -> torch.Tensor:
    """C[b, m] = <Y[b], psi_m> by the tensor-core contraction of the batched path (Eq. 9 for B <= 64 signals)."""
    p, N, M, ld = _dict_args(psi_t)
    dev = psi_t.device
    if not (Y.is_cuda and Y.dtype == torch.float32 and Y.dim() == 2 and Y.shape[1] == N and (N == 1 or Y.stride(1) == 1)):
        raise TypeError("Y must be a CUDA float32 [B, N] tensor with unit stride along N")
    B = Y.shape[0]
    ldy = Y.stride(0) if B > 1 else max(Y.stride(0), N)
    C_out = torch.empty(B, M, dtype=torch.float32, device=dev) if C_out is None else C_out
    need = lib.mp_correlate_batched_workspace_bytes(N, M, B)
    ws = torch.empty(need + 256, dtype=torch.uint8, device=dev)
    base = ws.data_ptr()
    off = (-base) % 256
    with torch.cuda.device(dev):
        _check(lib.mp_correlate_batched(p, N, M, ld, Y.data_ptr(), ldy, B, _dev(C_out, torch.float32, "C"),
                                        base + off, ws.numel() - off, _stream_ptr(stream)))
    C_out._mp_workspace = ws          # keep the workspace alive until the stream has run the kernel
    return C_out


def mp_encode_sparse(psi_t: torch.Tensor, idx: torch.Tensor, val: torch.Tensor, *, y=None, stream=None) -> torch.Tensor:
    """Eq. 2: y = Psi x for a K-sparse x given as (idx int32[K], val float32[K]) device tensors."""
    p, N, M, ld = _dict_args(psi_t)
    K = idx.numel()
    if val.numel() != K:
        raise ValueError("idx and val must have the same length")
    y = torch.empty(N, dtype=torch.float32, device=psi_t.device) if y is None else y
    with torch.cuda.device(psi_t.device):
        _check(lib.mp_encode_sparse(p, N, M, ld, _dev(idx, torch.int32, "idx") if K else None,
                                    _dev(val, torch.float32, "val") if K else None, K, _dev(y, torch.float32, "y"),
                                    _stream_ptr(stream)))
    return y


def mp_reconstruction_error(x_hat: torch.Tensor, x: torch.Tensor, *, out=None, stream=None) -> torch.Tensor:
    """Eq. 14: 100 * ||x_hat - x||^2 / ||x||^2 as a float64[1] device tensor."""
    if x_hat.numel() != x.numel():
        raise ValueError("x_hat and x must have the same length")
    out = torch.empty(1, dtype=torch.float64, device=x.device) if out is None else out
    with torch.cuda.device(x.device):
        _check(lib.mp_reconstruction_error(_dev(x_hat, torch.float32, "x_hat"), _dev(x, torch.float32, "x"), x.numel(),
                                           _dev(out, torch.float64, "err_pct"), _stream_ptr(stream)))
    return out


def _dict_args_f64(psi_t: torch.Tensor):
    if not (psi_t.is_cuda and psi_t.dtype == torch.float64 and psi_t.dim() == 2 and (psi_t.shape[1] == 1 or psi_t.stride(1) == 1)):
        raise TypeError("psi_t must be a CUDA float64 [M, N] tensor with unit stride along N (atom-major)")
    M, N = psi_t.shape
    ld = psi_t.stride(0) if M > 1 else max(psi_t.stride(0), N)
    return psi_t.data_ptr(), N, M, ld


def mp_normalize_columns_f64(psi_t: torch.Tensor, norms_out: torch.Tensor | None = None, stream=None) -> None:
    """Eq. 4 in float64, in place on the device tensor psi_t[M, N]."""
    p, N, M, ld = _dict_args_f64(psi_t)
    n = _dev(norms_out, torch.float64, "norms_out") if norms_out is not None else None
    with torch.cuda.device(psi_t.device):
        _check(lib.mp_normalize_columns_f64(p, N, M, ld, n, _stream_ptr(stream)))


def mp_recover_f64(psi_t: torch.Tensor, y: torch.Tensor, eps: float, max_iter: int, *, trace: bool = False,
                   workspace=None, stream=None) -> Recovered:
    """Eq. 8-12 in double precision (float64 dictionary, signal, coefficients and residual)."""
    p, N, M, ld = _dict_args_f64(psi_t)
    dev = psi_t.device
    if y.numel() != N:
        raise ValueError("y must have N elements")
    x = torch.empty(M, dtype=torch.float64, device=dev)
    r = torch.empty(N, dtype=torch.float64, device=dev)
    n_iter = torch.empty(1, dtype=torch.int32, device=dev)
    idx_trace = torch.empty(max(max_iter, 1), dtype=torch.int32, device=dev) if trace else None
    c_trace = torch.empty(max(max_iter, 1), dtype=torch.float64, device=dev) if trace else None
    need = lib.mp_workspace_bytes_f64(N, M)
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=dev)
    base = workspace.data_ptr()
    off = (-base) % 256
    with torch.cuda.device(dev):
        _check(lib.mp_recover_f64(p, N, M, ld, _dev(y, torch.float64, "y"), float(eps), int(max_iter),
                                  x.data_ptr(), r.data_ptr(), n_iter.data_ptr(),
                                  idx_trace.data_ptr() if trace else None, c_trace.data_ptr() if trace else None,
                                  base + off, workspace.numel() - off, _stream_ptr(stream)))
    return Recovered(x, r, n_iter, idx_trace, c_trace, workspace)


def mp_recover_omp(psi_t: torch.Tensor, y: torch.Tensor, eps: float, max_iter: int, *, trace: bool = False,
                   workspace=None, stream=None) -> Recovered:
    """Orthogonal MP: MP's selection + least-squares refit; outputs are device tensors."""
    p, N, M, ld = _dict_args(psi_t)
    dev = psi_t.device
    if y.numel() != N:
        raise ValueError("y must have N elements")
    x = torch.empty(M, dtype=torch.float32, device=dev)
    r = torch.empty(N, dtype=torch.float32, device=dev)
    n_iter = torch.empty(1, dtype=torch.int32, device=dev)
    idx_trace = torch.empty(max(min(max_iter, N), 1), dtype=torch.int32, device=dev) if trace else None
    need = lib.mp_workspace_bytes_omp(N, M, int(max_iter))
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=dev)
    base = workspace.data_ptr()
    off = (-base) % 256
    with torch.cuda.device(dev):
        _check(lib.mp_recover_omp(p, N, M, ld, _dev(y, torch.float32, "y"), float(eps), int(max_iter),
                                  x.data_ptr(), r.data_ptr(), n_iter.data_ptr(), idx_trace.data_ptr() if trace else None,
                                  base + off, workspace.numel() - off, _stream_ptr(stream)))
    return Recovered(x, r, n_iter, idx_trace, None, workspace)


def mp_pack_signs(psi_t: torch.Tensor, stream=None):
    """Sign bits of a +-scale (Bernoulli, Eq. 13) dictionary -> (bits int32[M, ldw], scale float, n_bad int).
    Synchronises to read scale and n_bad back (a one-off per dictionary)."""
    p, N, M, ld = _dict_args(psi_t)
    ldw = ((N + 31) // 32 + 3) // 4 * 4
    bits = torch.empty(M, ldw, dtype=torch.int32, device=psi_t.device)
    scale = torch.empty(1, dtype=torch.float32, device=psi_t.device)
    n_bad = torch.empty(1, dtype=torch.int32, device=psi_t.device)
    with torch.cuda.device(psi_t.device):
        _check(lib.mp_pack_signs(p, N, M, ld, bits.data_ptr(), ldw, scale.data_ptr(), n_bad.data_ptr(), _stream_ptr(stream)))
    return bits, float(scale.item()), int(n_bad.item())


def mp_recover_signs(bits: torch.Tensor, N: int, scale: float, y: torch.Tensor, eps: float, max_iter: int, *,
                     trace: bool = False, workspace=None, stream=None) -> Recovered:
    """Eq. 8-12 on a sign-packed Bernoulli dictionary (bits from mp_pack_signs)."""
    if not (bits.is_cuda and bits.dtype == torch.int32 and bits.dim() == 2 and bits.is_contiguous()):
        raise TypeError("bits must be a contiguous CUDA int32 [M, ldw] tensor")
    M, ldw = bits.shape
    dev = bits.device
    x = torch.empty(M, dtype=torch.float32, device=dev)
    r = torch.empty(N, dtype=torch.float32, device=dev)
    n_iter = torch.empty(1, dtype=torch.int32, device=dev)
    idx_trace = torch.empty(max(max_iter, 1), dtype=torch.int32, device=dev) if trace else None
    c_trace = torch.empty(max(max_iter, 1), dtype=torch.float32, device=dev) if trace else None
    workspace, wp, wb = _workspace(N, M, 1, workspace, dev)
    with torch.cuda.device(dev):
        _check(lib.mp_recover_signs(bits.data_ptr(), N, M, ldw, float(scale), _dev(y, torch.float32, "y"), float(eps), int(max_iter),
                                    x.data_ptr(), r.data_ptr(), n_iter.data_ptr(),
                                    idx_trace.data_ptr() if trace else None, c_trace.data_ptr() if trace else None,
                                    wp, wb, _stream_ptr(stream)))
    return Recovered(x, r, n_iter, idx_trace, c_trace, workspace)


def mp_recover_signs_many(bits: torch.Tensor, N: int, scale: float, Y: torch.Tensor, eps: float, max_iter: int, *,
                          trace: bool = False, workspace=None, stream=None) -> Recovered:
    """P independent problems on sign-packed Bernoulli dictionaries (the paper's Fig. 1 workload in its own representation):
    bits int32[P, M, ldw] (mp_pack_signs of the [P*M, N] stack, viewed per problem; [M, ldw] = one shared dictionary),
    Y[P, N] -> X[P, M], R[P, N], n_iter[P] (+ traces); one CTA per problem, the bits stationary in its shared memory."""
    if not (bits.is_cuda and bits.dtype == torch.int32 and bits.dim() in (2, 3) and bits.is_contiguous()):
        raise TypeError("bits must be a contiguous CUDA int32 [P, M, ldw] (or [M, ldw]) tensor")
    M, ldw = bits.shape[-2:]
    dev = bits.device
    if not (Y.is_cuda and Y.dtype == torch.float32 and Y.dim() == 2 and Y.shape[1] == N and (N == 1 or Y.stride(1) == 1)):
        raise TypeError("Y must be a CUDA float32 [P, N] tensor with unit stride along N")
    P = Y.shape[0]
    if bits.dim() == 3 and bits.shape[0] != P:
        raise ValueError("bits[P, M, ldw] and Y[P, N] disagree on P")
    pstride = M * ldw if bits.dim() == 3 else 0
    ldy = Y.stride(0) if P > 1 else max(Y.stride(0), N)
    X = torch.empty(P, M, dtype=torch.float32, device=dev)
    R = torch.empty(P, N, dtype=torch.float32, device=dev)
    n_iter = torch.empty(P, dtype=torch.int32, device=dev)
    ldt = max(max_iter, 1)
    idx_trace = torch.empty(P, ldt, dtype=torch.int32, device=dev) if trace else None
    c_trace = torch.empty(P, ldt, dtype=torch.float32, device=dev) if trace else None
    if workspace is None:
        workspace = torch.empty(lib.mp_workspace_bytes_signs_many(N, M, P) + 256, dtype=torch.uint8, device=dev)
    base = workspace.data_ptr()
    off = (-base) % 256
    with torch.cuda.device(dev):
        _check(lib.mp_recover_signs_many(bits.data_ptr(), N, M, ldw, pstride, float(scale), Y.data_ptr(), ldy, P, float(eps), int(max_iter),
                                         X.data_ptr(), R.data_ptr(), n_iter.data_ptr(),
                                         idx_trace.data_ptr() if trace else None, c_trace.data_ptr() if trace else None, ldt,
                                         base + off, workspace.numel() - off, _stream_ptr(stream)))
    return Recovered(X, R, n_iter, idx_trace, c_trace, workspace)


def _host(t: torch.Tensor, dtype, what: str):
    if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{what} must be a contiguous CPU {dtype} tensor")
    return t.data_ptr()


def _host_dict(t: torch.Tensor):
    if t.is_cuda or t.dtype != torch.float32 or t.dim() != 2 or not (t.shape[1] == 1 or t.stride(1) == 1):
        raise TypeError("psi_t must be a CPU float32 [M, N] tensor with unit stride along N")
    return t.data_ptr()


def mp_recover_host(psi_t: torch.Tensor, y: torch.Tensor, eps: float, max_iter: int, *, normalize: bool = False,
                    trace: bool = False, device: int = 0) -> Recovered:
    """HOST tensors in, HOST tensors out (copies, kernels and the final synchronise inside the C call)."""
    M, N = psi_t.shape
    x = torch.empty(M, dtype=torch.float32).pin_memory()
    r = torch.empty(N, dtype=torch.float32).pin_memory()
    n_iter = torch.zeros(1, dtype=torch.int32).pin_memory()
    it = torch.empty(max(max_iter, 1), dtype=torch.int32) if trace else None
    ct = torch.empty(max(max_iter, 1), dtype=torch.float32) if trace else None
    with torch.cuda.device(device):
        _check(lib.mp_recover_host(_host_dict(psi_t), N, M, psi_t.stride(0) if M > 1 else N,
                                   int(normalize), _host(y, torch.float32, "y"), float(eps), int(max_iter),
                                   x.data_ptr(), r.data_ptr(), n_iter.data_ptr(),
                                   it.data_ptr() if trace else None, ct.data_ptr() if trace else None))
    return Recovered(x, r, n_iter, it, ct, None)


def mp_recover_batched_host(psi_t: torch.Tensor, Y: torch.Tensor, eps: float, max_iter: int, *,
                            normalize: bool = False, device: int = 0) -> Recovered:
    M, N = psi_t.shape
    B = Y.shape[0]
    X = torch.empty(B, M, dtype=torch.float32).pin_memory()
    R = torch.empty(B, N, dtype=torch.float32).pin_memory()
    n_iter = torch.zeros(B, dtype=torch.int32).pin_memory()
    with torch.cuda.device(device):
        _check(lib.mp_recover_batched_host(_host_dict(psi_t), N, M, psi_t.stride(0) if M > 1 else N,
                                           int(normalize), _host(Y, torch.float32, "Y"), N, B, float(eps), int(max_iter),
                                           X.data_ptr(), R.data_ptr(), n_iter.data_ptr()))
    return Recovered(X, R, n_iter, None, None, None)


@dataclasses.dataclass
class Dictionary:
    """An mp_dictionary handle (the dictionary goes to the device once).  `psi_t` is a torch view of the device copy
    when the handle borrowed a device tensor (kept alive here), else None."""
    ptr: int
    N: int
    M: int
    ld: int
    device: int
    psi_ptr: int
    psi_t: torch.Tensor | None = None


def mp_dictionary_create(psi_t: torch.Tensor, *, normalize: bool = False) -> Dictionary:
    """psi_t[M, N] float32 on the HOST (uploaded, optionally normalised on the device; the host tensor is untouched) or on the
    DEVICE (borrowed; normalised in place if asked).  The handle lives on the current CUDA device / the tensor's device."""
    if not (psi_t.dtype == torch.float32 and psi_t.dim() == 2 and (psi_t.shape[1] == 1 or psi_t.stride(1) == 1)):
        raise TypeError("psi_t must be a float32 [M, N] tensor with unit stride along N (atom-major)")
    M, N = psi_t.shape
    ld = psi_t.stride(0) if M > 1 else max(psi_t.stride(0), N)
    out = _vp(None)
    dev = psi_t.device if psi_t.is_cuda else torch.device("cuda", torch.cuda.current_device())
    with torch.cuda.device(dev):
        if psi_t.is_cuda:
            torch.cuda.current_stream().synchronize()            # the handle works on its own stream
        _check(lib.mp_dictionary_create(psi_t.data_ptr(), 0 if psi_t.is_cuda else 1, N, M, ld, int(normalize), C.byref(out)))
    p = _vp(None)
    _check(lib.mp_dictionary_info(out, None, None, None, C.byref(p)))
    return Dictionary(out.value, N, M, ld, dev.index if dev.index is not None else 0, p.value, psi_t if psi_t.is_cuda else None)


def mp_dictionary_destroy(h: Dictionary) -> None:
    if h.ptr:
        _check(lib.mp_dictionary_destroy(h.ptr))
        h.ptr = 0
        h.psi_t = None


def mp_recover_host_h(h: Dictionary, y: torch.Tensor, eps: float, max_iter: int, *, trace: bool = False) -> Recovered:
    """mp_recover_host without the dictionary transfer: HOST y in, HOST x~, r, n_iter (and traces) out; synchronous."""
    x = torch.empty(h.M, dtype=torch.float32).pin_memory()
    r = torch.empty(h.N, dtype=torch.float32).pin_memory()
    n_iter = torch.zeros(1, dtype=torch.int32).pin_memory()
    it = torch.empty(max(max_iter, 1), dtype=torch.int32) if trace else None
    ct = torch.empty(max(max_iter, 1), dtype=torch.float32) if trace else None
    if y.numel() != h.N:
        raise ValueError("y must have N elements")
    _check(lib.mp_recover_host_h(h.ptr, _host(y, torch.float32, "y"), float(eps), int(max_iter), x.data_ptr(), r.data_ptr(),
                                 n_iter.data_ptr(), it.data_ptr() if trace else None, ct.data_ptr() if trace else None))
    return Recovered(x, r, n_iter, it, ct, None)


def mp_recover_batched_host_h(h: Dictionary, Y: torch.Tensor, eps: float, max_iter: int, *, trace: bool = False) -> Recovered:
    if Y.dim() != 2 or Y.shape[1] != h.N:
        raise ValueError("Y must be [B, N]")
    B = Y.shape[0]
    X = torch.empty(B, h.M, dtype=torch.float32).pin_memory()
    R = torch.empty(B, h.N, dtype=torch.float32).pin_memory()
    n_iter = torch.zeros(B, dtype=torch.int32).pin_memory()
    ldt = max(max_iter, 1)
    it = torch.empty(B, ldt, dtype=torch.int32) if trace else None
    ct = torch.empty(B, ldt, dtype=torch.float32) if trace else None
    _check(lib.mp_recover_batched_host_h(h.ptr, _host(Y, torch.float32, "Y"), h.N, B, float(eps), int(max_iter),
                                         X.data_ptr(), R.data_ptr(), n_iter.data_ptr(),
                                         it.data_ptr() if trace else None, ct.data_ptr() if trace else None, ldt))
    return Recovered(X, R, n_iter, it, ct, None)
