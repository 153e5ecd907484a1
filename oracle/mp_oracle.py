"""ctypes binding of the CPU oracle (oracle/mp_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only -- every number is computed by the C loops.  Dictionaries are
atom-major numpy arrays psi_t[M, N] (float64 -> *_f64 routines, float32 -> *_f32 routines,
which promote each element to double on the fly).
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

from . import build as _build

__all__ = ["normalize_columns", "correlate", "argmax_abs", "nrm2", "mp", "mp_replay",
           "mp_batched", "omp", "OMPResult", "encode_sparse", "atom_major_from_rowmajor", "reconstruction_error_pct", "MPResult", "ReplayResult", "default_threads"]

_lib = C.CDLL(_build.build())

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int)
_vp = C.c_void_p

_lib.oracle_nrm2.restype = C.c_double
_lib.oracle_nrm2.argtypes = [_vp, C.c_int]
_lib.oracle_argmax_abs.restype = C.c_int
_lib.oracle_argmax_abs.argtypes = [_vp, C.c_int]
_lib.oracle_normalize_columns_f64.restype = None
_lib.oracle_normalize_columns_f64.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp]
for _s in ("f64", "f32"):
    f = getattr(_lib, "oracle_correlate_" + _s)
    f.restype = None
    f.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, _vp, C.c_int]
    f = getattr(_lib, "oracle_mp_" + _s)
    f.restype = C.c_int
    f.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, C.c_double, C.c_int,
                  _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int]
    f = getattr(_lib, "oracle_mp_replay_" + _s)
    f.restype = C.c_int
    f.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, _vp, _vp, C.c_int,
                  _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int]
_lib.oracle_mp_batched_f32.restype = C.c_int
_lib.oracle_mp_batched_f32.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, C.c_int64, C.c_int,
                                       C.c_double, C.c_int, _vp, _vp, _vp, C.c_int]
_lib.oracle_omp_f32.restype = C.c_int
_lib.oracle_omp_f32.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, C.c_double, C.c_int, _vp, C.c_int,
                                _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int]
_lib.oracle_encode_sparse_f32.restype = C.c_int
_lib.oracle_encode_sparse_f32.argtypes = [_vp, C.c_int, C.c_int, C.c_int64, _vp, _vp, C.c_int, _vp]
_lib.oracle_reconstruction_error_pct.restype = C.c_double
_lib.oracle_reconstruction_error_pct.argtypes = [_vp, _vp, C.c_int]


def default_threads() -> int:
    return len(os.sched_getaffinity(0))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_vp)


def _psi(psi_t):
    """-> (array kept alive, suffix, N, M, ld)"""
    if psi_t.ndim != 2 or psi_t.strides[1] != psi_t.itemsize or psi_t.strides[0] % psi_t.itemsize:
        raise ValueError("psi_t must be [M, N] with unit stride along N")
    if psi_t.dtype == np.float64:
        s = "f64"
    elif psi_t.dtype == np.float32:
        s = "f32"
    else:
        raise TypeError("psi_t must be float64 or float32")
    M, N = psi_t.shape
    ld = psi_t.strides[0] // psi_t.itemsize
    if M == 1:
        ld = max(ld, N)          # a lone row's stride is arbitrary (numpy may report 0)
    return psi_t, s, N, M, ld


def _f64(v):
    return np.ascontiguousarray(v, dtype=np.float64)


def nrm2(v) -> float:
    v = _f64(v)
    return _lib.oracle_nrm2(_ptr(v), v.size)


def argmax_abs(c) -> int:
    c = _f64(c)
    return _lib.oracle_argmax_abs(_ptr(c), c.size)


def normalize_columns(psi_t):
    """Returns (normalised float64 copy [M, N], norms[M])."""
    out = np.array(psi_t, dtype=np.float64, order="C", copy=True)
    M, N = out.shape
    norms = np.empty(M, dtype=np.float64)
    _lib.oracle_normalize_columns_f64(_ptr(out), N, M, N, _ptr(norms))
    return out, norms


def correlate(psi_t, r, nthreads: int = 1):
    a, s, N, M, ld = _psi(psi_t)
    r = _f64(r)
    assert r.size == N
    c = np.empty(M, dtype=np.float64)
    getattr(_lib, "oracle_correlate_" + s)(_ptr(a), N, M, ld, _ptr(r), _ptr(c), nthreads)
    return c


@dataclasses.dataclass
class MPResult:
    x: np.ndarray        # [M] float64
    r: np.ndarray        # [N] float64
    n_iter: int
    idx: np.ndarray      # [n_iter] int32   atom chosen at iteration t
    c: np.ndarray        # [n_iter] float64 signed <r, psi_idx> added at iteration t
    gap: np.ndarray      # [n_iter] float64 relative top-two gap of |c| at iteration t
    rnorm: np.ndarray    # [n_iter+1] float64 ||r|| at the top of iteration t; last = final


def mp(psi_t, y, eps: float, max_iter: int, nthreads: int = 1) -> MPResult:
    a, s, N, M, ld = _psi(psi_t)
    y = _f64(y)
    assert y.size == N
    x = np.empty(M, dtype=np.float64)
    r = np.empty(N, dtype=np.float64)
    n_iter = C.c_int(0)
    idx = np.empty(max(max_iter, 1), dtype=np.int32)
    c = np.empty(max(max_iter, 1), dtype=np.float64)
    gap = np.empty(max(max_iter, 1), dtype=np.float64)
    rn = np.empty(max_iter + 1, dtype=np.float64)
    rc = getattr(_lib, "oracle_mp_" + s)(_ptr(a), N, M, ld, _ptr(y), float(eps), int(max_iter),
                                         _ptr(x), _ptr(r), C.byref(n_iter),
                                         _ptr(idx), _ptr(c), _ptr(gap), _ptr(rn), nthreads)
    if rc:
        raise ValueError("oracle_mp: invalid arguments")
    t = n_iter.value
    return MPResult(x, r, t, idx[:t].copy(), c[:t].copy(), gap[:t].copy(), rn[:t + 1].copy())


@dataclasses.dataclass
class ReplayResult:
    x: np.ndarray           # [M] state after the forced steps
    r: np.ndarray           # [N]
    argmax_ref: np.ndarray  # [t_run] the oracle's own argmax at step t
    cmax_ref: np.ndarray    # [t_run] max |c_ref| at step t
    c_at_idx: np.ndarray    # [t_run] signed c_ref at the imposed atom
    gap: np.ndarray         # [t_run] relative top-two gap of |c_ref|
    rnorm: np.ndarray       # [t_run+1]


def mp_replay(psi_t, y, idx_run, c_run=None, nthreads: int = 1) -> ReplayResult:
    a, s, N, M, ld = _psi(psi_t)
    y = _f64(y)
    idx_run = np.ascontiguousarray(idx_run, dtype=np.int32)
    t_run = idx_run.size
    if c_run is not None:
        c_run = _f64(c_run)
        assert c_run.size == t_run
    x = np.empty(M, dtype=np.float64)
    r = np.empty(N, dtype=np.float64)
    am = np.empty(max(t_run, 1), dtype=np.int32)
    cm = np.empty(max(t_run, 1), dtype=np.float64)
    ci = np.empty(max(t_run, 1), dtype=np.float64)
    gap = np.empty(max(t_run, 1), dtype=np.float64)
    rn = np.empty(t_run + 1, dtype=np.float64)
    rc = getattr(_lib, "oracle_mp_replay_" + s)(_ptr(a), N, M, ld, _ptr(y), _ptr(idx_run), _ptr(c_run), t_run,
                                                _ptr(x), _ptr(r), _ptr(am), _ptr(cm), _ptr(ci), _ptr(gap), _ptr(rn),
                                                nthreads)
    if rc:
        raise ValueError("oracle_mp_replay: invalid arguments")
    return ReplayResult(x, r, am[:t_run].copy(), cm[:t_run].copy(), ci[:t_run].copy(), gap[:t_run].copy(), rn)


def mp_batched(psi_t, Y, eps: float, max_iter: int, nthreads: int = 1):
    """Y[B, N] -> X[B, M], R[B, N], n_iter[B]  (float32 dictionary only)."""
    a, s, N, M, ld = _psi(psi_t)
    if s != "f32":
        raise TypeError("mp_batched takes the float32 dictionary")
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    B = Y.shape[0]
    X = np.empty((B, M), dtype=np.float64)
    R = np.empty((B, N), dtype=np.float64)
    n_iter = np.empty(B, dtype=np.int32)
    rc = _lib.oracle_mp_batched_f32(_ptr(a), N, M, ld, _ptr(Y), N, B, float(eps), int(max_iter),
                                    _ptr(X), _ptr(R), _ptr(n_iter), nthreads)
    if rc:
        raise ValueError("oracle_mp_batched: invalid arguments")
    return X, R, n_iter


@dataclasses.dataclass
class OMPResult:
    x: np.ndarray            # [M] float64: least-squares coefficients on the selected atoms, 0 elsewhere
    r: np.ndarray            # [N] float64: y - Psi_S x_S
    n_iter: int
    idx: np.ndarray          # [n_iter] atom taken at step t
    gap: np.ndarray          # [n_iter] relative top-two gap of |c| on the oracle's own r
    rnorm: np.ndarray        # [n_iter+1]
    argmax_ref: np.ndarray   # [n_iter] the oracle's own argmax (differs from idx only in a forced replay)
    cmax_ref: np.ndarray
    c_at_idx: np.ndarray
    status: int              # 0 ok, 2 = ended by a repeated atom / singular Gram matrix


def omp(psi_t, y, eps: float, max_iter: int, idx_force=None, nthreads: int = 1) -> OMPResult:
    """Orthogonal MP on the float32 dictionary; idx_force = teacher-forced replay of a given atom sequence."""
    a, s, N, M, ld = _psi(psi_t)
    if s != "f32":
        raise TypeError("omp takes the float32 dictionary")
    y = _f64(y)
    force = None if idx_force is None else np.ascontiguousarray(idx_force, dtype=np.int32)
    cap = max((force.size if force is not None else min(max_iter, N)), 1)
    x = np.empty(M); r = np.empty(N); n_iter = C.c_int(0)
    idx = np.empty(cap, dtype=np.int32); gap = np.empty(cap); rn = np.empty(cap + 1)
    am = np.empty(cap, dtype=np.int32); cm = np.empty(cap); ci = np.empty(cap)
    rc = _lib.oracle_omp_f32(_ptr(a), N, M, ld, _ptr(y), float(eps), int(max_iter),
                             _ptr(force) if force is not None else None, int(force.size) if force is not None else 0,
                             _ptr(x), _ptr(r), C.byref(n_iter), _ptr(idx), _ptr(gap), _ptr(rn), _ptr(am), _ptr(cm), _ptr(ci),
                             nthreads)
    if rc == 1:
        raise ValueError("oracle_omp: invalid arguments")
    t = n_iter.value
    return OMPResult(x, r, t, idx[:t].copy(), gap[:t].copy(), rn[:t + 1].copy(), am[:t].copy(), cm[:t].copy(), ci[:t].copy(), rc)


def encode_sparse(psi_t, idx, val) -> np.ndarray:
    """Eq. 2: y[n] = sum_k val[k] * Psi[n][idx[k]] (ascending k, float64) from the float32 dictionary."""
    a, s, N, M, ld = _psi(psi_t)
    if s != "f32":
        raise TypeError("encode_sparse takes the float32 dictionary")
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    val = _f64(val)
    assert idx.size == val.size
    y = np.empty(N, dtype=np.float64)
    if _lib.oracle_encode_sparse_f32(_ptr(a), N, M, ld, _ptr(idx), _ptr(val), int(idx.size), _ptr(y)):
        raise ValueError("oracle_encode_sparse: invalid arguments")
    return y


def reconstruction_error_pct(x_hat, x) -> float:
    x_hat, x = _f64(x_hat), _f64(x)
    return _lib.oracle_reconstruction_error_pct(_ptr(x_hat), _ptr(x), x.size)


def atom_major_from_rowmajor(psi) -> np.ndarray:
    """The paper's listings store Psi row-major, psi[n*M + m] (A2 P:360: `h_Psi[n*M + m]`); every routine here takes the
    atom-major psi_t[m, n] = Psi[n, m].  The definition written out, element by element (no arithmetic)."""
    psi = np.asarray(psi)
    N, M = psi.shape
    out = np.empty((M, N), dtype=psi.dtype)
    for n in range(N):
        out[:, n] = psi[n, :]
    return out
