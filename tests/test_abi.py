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
