"""CPU-side checks of the C-ABI boundary: the library loads without a GPU and exports every symbol
include/mp_b200.h declares; argument validation happens on the host before any CUDA work."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mp_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"MP_API\s+[\w\s\*]+?\b(mp_\w+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    from paper_0809_1833_b200 import build
    lib = C.CDLL(build.build())
    names = declared_symbols()
    assert len(names) >= 10 and "mp_recover" in names and "mp_recover_batched" in names and "mp_normalize_columns" in names
    for n in names:
        assert hasattr(lib, n), n


def test_workspace_bytes_and_knobs_without_gpu():
    import paper_0809_1833_b200 as mp
    assert mp.mp_workspace_bytes(0, 10, 1) == 0 and mp.mp_workspace_bytes(10, 10, 0) == 0
    a = mp.mp_workspace_bytes(4096, 16384, 1)
    b = mp.mp_workspace_bytes(4096, 16384, 2)
    assert a >= 8 * 16384 + 12 * 4096 and b > a and a % 256 == 0
    mp.mp_set_int("chunk", 32)
    assert mp.mp_get_int("chunk") == 32
    mp.mp_set_int("chunk", 64)
    with pytest.raises(mp.MPError) as e:
        mp.mp_set_int("no_such_knob", 1)
    assert e.value.status == mp.MP_ERR_INVALID_ARG and "no_such_knob" in mp.mp_last_error()


def test_argument_errors_are_detected_before_any_cuda_call():
    """Null pointers, bad sizes and misalignment return MP_ERR_INVALID_ARG / MP_ERR_WORKSPACE on a box with no GPU."""
    from paper_0809_1833_b200.binding import lib
    ok_ptr = C.c_void_p(4096)          # never dereferenced: validation fails first
    f = lib.mp_recover
    assert f(None, 8, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 0, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 8, 8, 6, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1   # ld < N
    assert f(ok_ptr, 6, 8, 6, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1   # ld % 4
    assert f(C.c_void_p(4100), 8, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 8, 8, 8, ok_ptr, -1.0, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 8, 8, 8, ok_ptr, float("nan"), 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 8, 8, 8, ok_ptr, 0.1, -1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 1 << 20, None) == 1
    assert f(ok_ptr, 8, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, None, 1 << 20, None) == 4
    assert f(ok_ptr, 8, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, ok_ptr, 16, None) == 4
    assert f(ok_ptr, 8, 8, 8, ok_ptr, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, None, None, C.c_void_p(4096 + 64), 1 << 20, None) == 4
    g = lib.mp_recover_batched
    assert g(ok_ptr, 8, 8, 8, ok_ptr, 8, 0, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 1          # B < 1
    assert g(ok_ptr, 8, 8, 8, ok_ptr, 4, 2, 0.1, 1, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 1          # ldy < N
    assert lib.mp_normalize_columns(None, 8, 8, 8, None, None) == 1
    assert lib.mp_last_error() != b""


def test_argument_errors_of_the_widened_entry_points():
    """encode / score / float64 / Orthogonal MP / batched correlation: validation happens on the host before any CUDA call."""
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    assert lib.mp_encode_sparse(None, 8, 8, 8, ok, ok, 2, ok, None) == 1
    assert lib.mp_encode_sparse(ok, 8, 8, 8, None, ok, 2, ok, None) == 1                      # K > 0 needs idx
    assert lib.mp_encode_sparse(ok, 8, 8, 8, ok, ok, -1, ok, None) == 1
    assert lib.mp_reconstruction_error(ok, ok, 0, ok, None) == 1
    assert lib.mp_reconstruction_error(ok, ok, 8, C.c_void_p(4100), None) == 1                # err_pct alignment
    f = lib.mp_recover_f64
    assert f(None, 8, 8, 8, ok, 0.1, 1, ok, ok, ok, None, None, ok, 1 << 20, None) == 1
    assert f(ok, 8, 8, 7, ok, 0.1, 1, ok, ok, ok, None, None, ok, 1 << 20, None) == 1           # ld < N
    assert f(ok, 7, 8, 7, ok, 0.1, 1, ok, ok, ok, None, None, ok, 1 << 20, None) == 1           # ld odd
    assert f(ok, 8, 8, 8, ok, -0.1, 1, ok, ok, ok, None, None, ok, 1 << 20, None) == 1
    assert f(ok, 8, 8, 8, ok, 0.1, 1, ok, ok, ok, None, None, ok, 16, None) == 4
    assert lib.mp_workspace_bytes_f64(0, 8) == 0 and lib.mp_workspace_bytes_f64(8, 8) >= 256 + 64
    g = lib.mp_recover_omp
    assert g(None, 8, 8, 8, ok, 0.1, 1, ok, ok, ok, None, ok, 1 << 20, None) == 1
    assert g(ok, 8, 8, 6, ok, 0.1, 1, ok, ok, ok, None, ok, 1 << 20, None) == 1               # ld < N
    assert g(ok, 8, 8, 8, ok, 0.1, -1, ok, ok, ok, None, ok, 1 << 20, None) == 1
    assert g(ok, 8, 8, 8, ok, 0.1, 4, ok, ok, ok, None, ok, 16, None) == 4
    a = lib.mp_workspace_bytes_omp(4096, 16384, 512)
    assert a >= 8 * 512 * 4096 and lib.mp_workspace_bytes_omp(4096, 16384, 10 ** 6) == lib.mp_workspace_bytes_omp(4096, 16384, 4096)
    h = lib.mp_correlate_batched
    assert h(ok, 8, 8, 8, ok, 8, 65, ok, ok, 1 << 20, None) == 1                              # B > 64
    assert h(ok, 8, 8, 8, ok, 8, 2, ok, ok, 16, None) == 4
    assert lib.mp_correlate_batched_workspace_bytes(8, 8, 65) == 0


def test_argument_errors_of_mp_recover_many():
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    f = lib.mp_recover_many
    good = dict(psi=ok, N=8, M=8, ld=8, ps=64, Y=ok, ldy=8, P=2, eps=0.1, T=4, X=ok, R=ok, n=ok, it=None, ct=None, ldt=4, ws=ok, wsb=1 << 20)

    def call(**kw):
        a = dict(good, **kw)
        return f(a["psi"], a["N"], a["M"], a["ld"], a["ps"], a["Y"], a["ldy"], a["P"], a["eps"], a["T"], a["X"], a["R"], a["n"],
                 a["it"], a["ct"], a["ldt"], a["ws"], a["wsb"], None)
    assert call(psi=None) == 1 and call(P=0) == 1 and call(ps=32) == 1 and call(ps=66) == 1        # stride < M*ld, stride % 4
    assert call(ldy=4) == 1 and call(T=-1) == 1 and call(eps=-1.0) == 1 and call(Y=None) == 1
    assert call(it=ok, ldt=2) == 1                                                                # ldt < max_iter
    assert call(ws=None) == 4 and call(wsb=16) == 4
    assert lib.mp_workspace_bytes_many(8, 8, 0) == 0 and lib.mp_workspace_bytes_many(8, 8, 3) >= 256


def test_argument_errors_of_mp_transpose_rowmajor():
    from paper_0809_1833_b200.binding import lib
    ok, ok2 = C.c_void_p(4096), C.c_void_p(1 << 30)
    f = lib.mp_transpose_rowmajor
    assert f(None, 8, 8, 8, ok2, 8, None) == 1 and f(ok, 8, 8, 8, None, 8, None) == 1
    assert f(ok, 8, 8, 7, ok2, 8, None) == 1                                   # ldr < M
    assert f(ok, 8, 8, 8, ok2, 6, None) == 1                                   # ld < N / ld % 4
    assert f(ok, 8, 8, 8, C.c_void_p(4096 + 64), 8, None) == 1                 # overlapping buffers


def test_argument_errors_of_mp_recover_signs_many():
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    f = lib.mp_recover_signs_many

    def call(bits=ok, N=64, M=8, ldw=2, ps=16, scale=0.125, Y=ok, ldy=64, P=2, eps=0.1, T=4, X=ok, R=ok, n=ok, it=None, ct=None, ldt=4, ws=ok, wsb=256):
        return f(bits, N, M, ldw, ps, scale, Y, ldy, P, eps, T, X, R, n, it, ct, ldt, ws, wsb, None)
    assert call(bits=None) == 1 and call(P=0) == 1 and call(ldw=1) == 1 and call(ps=8) == 1 and call(scale=0.0) == 1
    assert call(ldy=32) == 1 and call(T=-1) == 1 and call(eps=float("nan")) == 1 and call(it=ok, ldt=2) == 1
    assert call(ws=None) == 4 and call(wsb=16) == 4
    assert lib.mp_workspace_bytes_signs_many(8, 8, 0) == 0 and lib.mp_workspace_bytes_signs_many(8, 8, 3) == 256


def test_argument_errors_of_the_dictionary_handle():
    """mp_dictionary_create / *_host_h validate on the host before any CUDA call; destroying NULL is allowed."""
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    out = C.c_void_p(None)
    f = lib.mp_dictionary_create
    assert f(None, 1, 8, 8, 8, 0, C.byref(out)) == 1 and out.value is None
    assert f(ok, 1, 0, 8, 8, 0, C.byref(out)) == 1 and f(ok, 1, 8, 0, 8, 0, C.byref(out)) == 1
    assert f(ok, 1, 8, 8, 6, 0, C.byref(out)) == 1 and f(ok, 0, 6, 8, 6, 0, C.byref(out)) == 1       # ld < N; device ld % 4
    assert f(C.c_void_p(4100), 0, 8, 8, 8, 0, C.byref(out)) == 1                                     # misaligned device pointer
    assert f(ok, 1, 8, 8, 8, 0, None) == 1
    assert lib.mp_dictionary_destroy(None) == 0
    assert lib.mp_dictionary_info(None, None, None, None, None) == 1
    assert lib.mp_recover_host_h(None, ok, 0.1, 1, ok, ok, ok, None, None) == 1
    assert lib.mp_recover_batched_host_h(None, ok, 8, 1, 0.1, 1, ok, ok, ok, None, None, 1) == 1
    assert b"handle" in lib.mp_last_error()


def test_concurrent_builds_are_serialised_and_the_waiter_does_not_rebuild(monkeypatch):
    """Ranks / xdist workers that import the package at the same moment: one compiles under the lock on build/.lock, the others
    wait and then find the library up to date (paper_0809_1833_b200/build.py).  The compile is replaced by a stub here."""
    import threading
    import time
    from paper_0809_1833_b200 import build as B
    state = {"built": 0, "inside": 0, "overlap": False}

    def fake_build(verbose):
        state["inside"] += 1
        state["overlap"] |= state["inside"] > 1
        time.sleep(0.3)
        state["built"] += 1
        state["inside"] -= 1
        return B.LIB

    monkeypatch.setattr(B, "_build_locked", fake_build)
    monkeypatch.setattr(B, "_up_to_date", lambda: state["built"] > 0)
    threads = [threading.Thread(target=B.build) for _ in range(3)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert state["built"] == 1 and not state["overlap"]
    state["built"] = 0
    threads = [threading.Thread(target=B.build, kwargs={"force": True}) for _ in range(2)]     # forced: both build, one after the other
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert state["built"] == 2 and not state["overlap"]


def test_probe_read_argument_errors_without_gpu():
    """mp_probe_read validates on the host: null / misaligned buffer, passes < 1."""
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    n = C.c_ulonglong(0)
    assert lib.mp_probe_read(None, 1 << 24, 1, ok, C.byref(n), None) == 1
    assert lib.mp_probe_read(ok, 1 << 24, 1, None, C.byref(n), None) == 1
    assert lib.mp_probe_read(C.c_void_p(4100), 1 << 24, 1, ok, C.byref(n), None) == 1
    assert lib.mp_probe_read(ok, 1 << 24, 0, ok, C.byref(n), None) == 1
