"""mp_recover_noalloc: the solver for callers that cannot allocate device memory.

Some users of this library run inside a process that is not theirs: a plug-in of a server or framework whose own memory pool
has taken the whole GPU (cudaMalloc fails, or is against the host's rules), or a loop with a latency bound that an allocation
could break by stalling the device.  They cannot make the `workspace` every other solver asks for.  mp_recover_noalloc takes
inputs and outputs only and keeps its scratch (256 B of control words + M float64 coefficients) in a fixed 512.25 KiB array
inside the library, so it serves M <= MP_NOALLOC_MAX_M = 65536 and refuses anything larger.

What is checked here:
  * the limit and the argument rules, on the host, without a GPU (nothing is enqueued before they pass);
  * on a GPU, that two calls IN A ROW on one stream -- no synchronisation between them, different signals, so the second call
    finds the array as the first one left it -- give exactly what mp_recover gives on the same inputs with a caller-made
    workspace and the same kernel (knob "algo" = 3).  It is the same arithmetic in the same order, so the comparison is
    bit for bit, which is also what the repository's other same-kernel comparisons use; one result is graded against the
    float64 oracle as well.  A large-M call precedes a small-M one so that left-over coefficients would show;
  * that no-alloc calls enqueued on a side stream either side of an ordinary workspace solve, with no host synchronisation in
    between, each still give the bits of the same solve done alone: order on the GPU is all that keeps calls apart.

This file is named to be collected last (pytest -x stops at the first failure, and a failure here must not hide the parity
tests), and it does not depend on what ran before it: it sets the one knob it needs and puts it back.
"""
import ctypes as C

import numpy as np
import pytest

import problems


def test_limit_and_argument_errors_are_reported_on_the_host():
    """M beyond the built-in array -> MP_ERR_UNSUPPORTED with the limit in the message; bad arguments -> MP_ERR_INVALID_ARG.
    The pointers are fakes that are never dereferenced: every check happens before the first CUDA call."""
    import paper_0809_1833_b200 as mp
    from paper_0809_1833_b200.binding import lib
    ok = C.c_void_p(4096)
    f = lib.mp_recover_noalloc
    limit = mp.MP_NOALLOC_MAX_M
    assert limit == 65536
    assert f(ok, 8, limit + 1, 8, ok, 0.1, 1, ok, ok, ok, None, None, None) == mp.MP_ERR_UNSUPPORTED
    msg = mp.mp_last_error()
    assert str(limit) in msg and "mp_recover" in msg
    assert f(None, 8, 8, 8, ok, 0.1, 1, ok, ok, ok, None, None, None) == mp.MP_ERR_INVALID_ARG
    assert f(ok, 8, 8, 6, ok, 0.1, 1, ok, ok, ok, None, None, None) == mp.MP_ERR_INVALID_ARG          # ld < N
    assert f(C.c_void_p(4100), 8, 8, 8, ok, 0.1, 1, ok, ok, ok, None, None, None) == mp.MP_ERR_INVALID_ARG
    assert f(ok, 8, 8, 8, ok, 0.1, 1, ok, None, ok, None, None, None) == mp.MP_ERR_INVALID_ARG         # r missing
    assert f(ok, 8, 8, 8, ok, float("nan"), 1, ok, ok, ok, None, None, None) == mp.MP_ERR_INVALID_ARG
    assert f(ok, 8, 8, 8, ok, 0.1, -1, ok, ok, ok, None, None, None) == mp.MP_ERR_INVALID_ARG


def _workspace_path(mp, torch, psi_d, y_d, eps, T):
    """The existing path: mp_recover with a caller-made workspace, on the register-streaming kernel."""
    mp.mp_set_int("algo", 3)
    try:
        res = mp.mp_recover(psi_d, y_d, eps, T, trace=True)
        torch.cuda.synchronize()
        assert mp.mp_get_int("info_algo") == 3
    finally:
        mp.mp_set_int("algo", 0)
    t = int(res.n_iter.item())
    return res.x.cpu().numpy(), res.r.cpu().numpy(), t, res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t]


# (N, M, K): the largest M the array holds (with left-over coefficients for the next case to trip over), a ragged shape
# (N % 4 != 0, M not a multiple of the grid), and a shape whose rows span several chunks per atom
SHAPES = [(64, 65536, 6), (515, 700, 10), (1024, 4096, 24)]


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path():
    import torch
    import grading
    import paper_0809_1833_b200 as mp

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    launches_before = mp.mp_launch_count()
    graded = False
    for N, M, K in SHAPES:
        T = 3 * K + 2
        pb = problems.make_problem(problems.custom_config(N, M, K, eps=1e-5, max_iter=T, B=2), seed=N + M)
        ld = (N + 3) // 4 * 4
        buf = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")       # pad columns hold garbage on purpose
        buf[:, :N] = torch.from_numpy(pb.psi32).cuda()
        psi_d = buf[:, :N]
        ys = [torch.from_numpy(np.ascontiguousarray(pb.Y[b])).cuda() for b in range(2)]
        want = [_workspace_path(mp, torch, psi_d, ys[b], pb.cfg.eps, T) for b in range(2)]
        assert want[0][2] > 0 and want[1][2] > 0 and not np.array_equal(want[0][3], want[1][3])   # two different solves

        # outputs made by the caller up front, as a caller that cannot allocate would have them; filled with a pattern
        outs = [dict(x=torch.full((M,), 3.0, device="cuda"), r=torch.full((N,), 3.0, device="cuda"),
                     n_iter=torch.full((1,), -7, dtype=torch.int32, device="cuda"),
                     idx_trace=torch.full((T,), -1, dtype=torch.int32, device="cuda"),
                     c_trace=torch.full((T,), 3.0, device="cuda")) for _ in range(2)]
        torch.cuda.synchronize()
        for b in range(2):                                                        # back to back, nothing in between
            mp.mp_recover_noalloc(psi_d, ys[b], pb.cfg.eps, T, **outs[b])
        torch.cuda.synchronize()

        for b in range(2):
            x, r, t, idx, c = want[b]
            o = outs[b]
            assert int(o["n_iter"].item()) == t, (N, M, b)
            assert np.array_equal(o["idx_trace"].cpu().numpy()[:t], idx), (N, M, b)
            assert np.array_equal(o["c_trace"].cpu().numpy()[:t], c), (N, M, b)
            assert np.array_equal(o["x"].cpu().numpy(), x), (N, M, b)
            assert np.array_equal(o["r"].cpu().numpy(), r), (N, M, b)
        if not graded and M <= 4096:                                              # and once against the float64 oracle
            o = outs[1]
            t = int(o["n_iter"].item())
            grading.grade_single(pb.psi32, pb.Y[1], pb.cfg.eps, T, o["x"].cpu().numpy(), o["r"].cpu().numpy(), t,
                                 o["idx_trace"].cpu().numpy()[:t], o["c_trace"].cpu().numpy()[:t])
            graded = True
    assert graded
    assert mp.mp_launch_count() - launches_before == 4 * len(SHAPES)             # every call above launched its kernel


@pytest.mark.gpu
def test_calls_ordered_on_a_side_stream_do_not_disturb_each_other():
    """The built-in array is shared by every call on the device, so what keeps calls apart is their order on the GPU.  Here a
    side stream carries: a no-alloc solve, a workspace solve of another signal, and a no-alloc solve of a third -- enqueued
    without a host synchronisation in between.  Stream order is all the entry point asks for: each result must be the bits of
    the same solve done on its own."""
    import torch
    import paper_0809_1833_b200 as mp

    N, M, K = 250, 1200, 8
    T = 3 * K + 2
    pb = problems.make_problem(problems.custom_config(N, M, K, eps=1e-5, max_iter=T, B=3), seed=41)
    ld = (N + 3) // 4 * 4
    buf = torch.zeros((M, ld), dtype=torch.float32, device="cuda")
    buf[:, :N] = torch.from_numpy(pb.psi32).cuda()
    psi_d = buf[:, :N]
    ys = [torch.from_numpy(np.ascontiguousarray(pb.Y[b])).cuda() for b in range(3)]
    want = [_workspace_path(mp, torch, psi_d, ys[b], pb.cfg.eps, T) for b in range(3)]

    def outputs():
        return dict(x=torch.empty(M, device="cuda"), r=torch.empty(N, device="cuda"),
                    n_iter=torch.empty(1, dtype=torch.int32, device="cuda"),
                    idx_trace=torch.empty(T, dtype=torch.int32, device="cuda"), c_trace=torch.empty(T, device="cuda"))

    outs = [outputs() for _ in range(3)]
    ws = torch.empty(mp.mp_workspace_bytes(N, M, 1) + 256, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    mp.mp_set_int("algo", 3)
    try:
        mp.mp_recover_noalloc(psi_d, ys[0], pb.cfg.eps, T, stream=side, **outs[0])
        mp.mp_recover(psi_d, ys[1], pb.cfg.eps, T, workspace=ws, stream=side, **outs[1])
        mp.mp_recover_noalloc(psi_d, ys[2], pb.cfg.eps, T, stream=side, **outs[2])
    finally:
        mp.mp_set_int("algo", 0)
    side.synchronize()
    for b in range(3):
        x, r, t, idx, c = want[b]
        o = outs[b]
        assert int(o["n_iter"].item()) == t, b
        assert np.array_equal(o["idx_trace"].cpu().numpy()[:t], idx) and np.array_equal(o["c_trace"].cpu().numpy()[:t], c), b
        assert np.array_equal(o["x"].cpu().numpy(), x) and np.array_equal(o["r"].cpu().numpy(), r), b
