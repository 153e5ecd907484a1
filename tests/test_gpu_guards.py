"""Guard-band tests (-m gpu): out-of-bounds WRITES of the CUDA path, found without a memory checker.

compute-sanitizer is closed on this GPU pool ("runs under it have left GPUs needing a reset"; profiles/sanitizer_r02.md),
so the library's stores are fenced in by hand: every caller-owned buffer a call may write (x~, r, n_iter, traces, workspace)
is the interior of a larger allocation whose margins hold a byte pattern, ragged shapes are used so that every kernel's
tail handling runs, and after the call the margins must be untouched and the read-only inputs (dictionary, signals)
unchanged.  The results themselves are graded by the parity tests; this file only looks at what must NOT change.
"""
import numpy as np
import pytest
import torch

import problems

pytestmark = pytest.mark.gpu

GUARD = 8192          # bytes on each side
PATTERN = 0xA5


@pytest.fixture(scope="module")
def mp():
    import paper_0809_1833_b200 as m
    yield m
    for k in ("algo", "batched_algo", "omp_algo", "grid"):
        m.mp_set_int(k, 0)


class Fenced:
    """`nbytes` of device memory, 256-byte aligned, between two pattern-filled margins."""

    def __init__(self, nbytes: int):
        self.n = (int(nbytes) + 255) // 256 * 256
        self.raw = torch.full((self.n + 2 * GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
        self.inner = self.raw[GUARD:GUARD + self.n]
        assert self.inner.data_ptr() % 256 == 0

    def view(self, dtype, count):
        return self.inner[: count * torch.empty(0, dtype=dtype).element_size()].view(dtype)

    def intact(self) -> bool:
        lo, hi = self.raw[:GUARD], self.raw[GUARD + self.n:]
        return bool((lo == PATTERN).all().item()) and bool((hi == PATTERN).all().item())


def padded(a: np.ndarray, ld: int, full: bool = False):
    """rows of `a` on the device with row stride ld (pads NaN)"""
    t = torch.full((a.shape[0], ld), float("nan"), dtype=torch.from_numpy(a).dtype, device="cuda")
    t[:, : a.shape[1]] = torch.from_numpy(a).cuda()
    return (t[:, : a.shape[1]], t) if full else t[:, : a.shape[1]]


SHAPES = [(250, 333, 6), (37, 1000, 4), (130, 2500, 8), (1, 5, 1), (515, 700, 10), (1030, 300, 12)]


@pytest.mark.parametrize("algo", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("N,M,K", SHAPES)
def test_single_signal_solvers_write_only_what_they_own(mp, N, M, K, algo):
    pb = problems.make_problem(problems.custom_config(N, M, K, eps=1e-5, max_iter=3 * K + 2), seed=N + M)
    T = pb.cfg.max_iter
    psi, psi_full = padded(pb.psi32, (N + 3) // 4 * 4 + 4, full=True)
    psi_before = psi.clone()
    y = torch.from_numpy(pb.Y[0]).cuda(); y_before = y.clone()
    fx, fr, fn, fi, fc = Fenced(4 * M), Fenced(4 * N), Fenced(4), Fenced(4 * T), Fenced(4 * T)
    fw = Fenced(mp.mp_workspace_bytes(N, M, 1))   # exactly the declared size: the fence starts where the workspace ends
    mp.mp_set_int("algo", algo)
    try:
        res = mp.mp_recover(psi, y, pb.cfg.eps, T, x=fx.view(torch.float32, M), r=fr.view(torch.float32, N),
                            n_iter=fn.view(torch.int32, 1), idx_trace=fi.view(torch.int32, T), c_trace=fc.view(torch.float32, T),
                            trace=True, workspace=fw.inner)
    except mp.MPError as e:
        if e.status == mp.MP_ERR_UNSUPPORTED:
            pytest.skip(str(e))
        raise
    torch.cuda.synchronize()
    assert 0 < int(res.n_iter.item()) <= T
    for name, f in (("x", fx), ("r", fr), ("n_iter", fn), ("idx_trace", fi), ("c_trace", fc), ("workspace", fw)):
        assert f.intact(), f"write outside {name}"
    assert torch.equal(psi, psi_before) and torch.equal(y, y_before), "a read-only input was modified"
    assert bool(torch.isnan(psi_full[:, N:]).all().item()), "dictionary pads were written"


@pytest.mark.parametrize("algo", [0, 1, 2, 3])
@pytest.mark.parametrize("N,M,K,B", [(250, 3000, 8, 5), (200, 1500, 6, 64), (515, 2100, 10, 3), (130, 4100, 5, 70)])
def test_batched_solvers_write_only_what_they_own(mp, N, M, K, B, algo):
    pb = problems.make_problem(problems.custom_config(N, M, K, eps=1e-5, max_iter=3 * K + 2, B=B), seed=N + B)
    T = pb.cfg.max_iter
    psi = padded(pb.psi32, (N + 3) // 4 * 4 + 4); psi_before = psi.clone()
    Y = padded(pb.Y, (N + 3) // 4 * 4); Y_before = Y.clone()
    fX, fR, fn, fi, fc = Fenced(4 * B * M), Fenced(4 * B * N), Fenced(4 * B), Fenced(4 * B * T), Fenced(4 * B * T)
    fw = Fenced(mp.mp_workspace_bytes(N, M, B))
    mp.mp_set_int("batched_algo", algo)
    try:
        res = mp.mp_recover_batched(psi, Y, pb.cfg.eps, T, X=fX.view(torch.float32, B * M).view(B, M),
                                    R=fR.view(torch.float32, B * N).view(B, N), n_iter=fn.view(torch.int32, B),
                                    idx_trace=fi.view(torch.int32, B * T).view(B, T), c_trace=fc.view(torch.float32, B * T).view(B, T),
                                    trace=True, workspace=fw.inner)
    except mp.MPError as e:
        if e.status == mp.MP_ERR_UNSUPPORTED:
            pytest.skip(str(e))
        raise
    torch.cuda.synchronize()
    assert int(res.n_iter.min().item()) > 0
    for name, f in (("X", fX), ("R", fR), ("n_iter", fn), ("idx_trace", fi), ("c_trace", fc), ("workspace", fw)):
        assert f.intact(), f"write outside {name}"
    assert torch.equal(psi, psi_before) and torch.equal(Y.nan_to_num(), Y_before.nan_to_num()), "a read-only input was modified"


@pytest.mark.parametrize("N,M,K", [(250, 333, 6), (130, 2500, 8), (515, 700, 10)])
def test_workspaces_of_the_widened_entry_points_are_respected(mp, N, M, K):
    """mp_recover_f64, mp_recover_omp (both drivers), mp_recover_many (shared and private dictionaries): the workspace each
    asks for is enough -- nothing is written past it -- and the dictionary is left alone."""
    pb = problems.make_problem(problems.custom_config(N, M, K, eps=1e-5, max_iter=2 * K, B=3), seed=7 * N)
    T = pb.cfg.max_iter
    lib = mp.binding.lib
    psi = padded(pb.psi32, (N + 3) // 4 * 4 + 4); psi_before = psi.clone()
    y = torch.from_numpy(pb.Y[0]).cuda()
    fw = Fenced(lib.mp_workspace_bytes_omp(N, M, T))
    for omp_algo in (1, 2):
        mp.mp_set_int("omp_algo", omp_algo)
        try:
            mp.mp_recover_omp(psi, y, pb.cfg.eps, T, trace=True, workspace=fw.inner)
        except mp.MPError as e:
            assert e.status == mp.MP_ERR_UNSUPPORTED
        torch.cuda.synchronize()
        assert fw.intact(), f"mp_recover_omp (omp_algo {omp_algo}) wrote outside its workspace"
    mp.mp_set_int("omp_algo", 0)
    psi64 = padded(pb.psi32.astype(np.float64), (N + 1) // 2 * 2 + 2); psi64_before = psi64.clone()
    fw = Fenced(lib.mp_workspace_bytes_f64(N, M))
    mp.mp_recover_f64(psi64, y.double(), pb.cfg.eps, T, trace=True, workspace=fw.inner)
    torch.cuda.synchronize()
    assert fw.intact(), "mp_recover_f64 wrote outside its workspace"
    assert torch.equal(psi64.nan_to_num(), psi64_before.nan_to_num())
    Y = padded(pb.Y, (N + 3) // 4 * 4)
    fw = Fenced(lib.mp_workspace_bytes_many(N, M, 3))
    try:
        mp.mp_recover_many(psi, Y, pb.cfg.eps, T, trace=True, workspace=fw.inner)
        torch.cuda.synchronize()
        assert fw.intact(), "mp_recover_many wrote outside its workspace"
    except mp.MPError as e:
        assert e.status == mp.MP_ERR_UNSUPPORTED
    assert torch.equal(psi, psi_before)
