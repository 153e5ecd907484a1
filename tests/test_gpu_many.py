"""GPU parity of mp_recover_many (many small independent problems, one thread-block cluster per
problem; the paper's Fig. 1 workload).  Problem q's result must equal a single-signal MP run on (dictionary q,
Y[q]): every problem is graded against the float64 oracle with the full contract of tests/grading.py (picks, step values,
residual, coefficients, stop rule).  The dot products are computed in the same order whatever the cluster size and whether
the dictionary is stationary in shared memory or streamed from L2, so those variants must agree bit for bit."""
import numpy as np
import pytest
import torch

import oracle
from paper_0809_1833_b200 import synth
import grading
import problems

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mp():
    import paper_0809_1833_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    yield m
    for k in ("many_cluster", "many_threads", "many_stat"):
        m.mp_set_int(k, 0)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_many(N, M, K, P, seed0=1, dictionary="gaussian", values="normal", eps=1e-5, max_iter=None):
    cfg = problems.custom_config(N, M, K, dictionary=dictionary, values=values, eps=eps, max_iter=max_iter)
    pbs = [problems.make_problem(cfg, seed0 + q) for q in range(P)]
    return cfg, pbs


def run_many(mp, pbs, eps, max_iter, ld=None, cluster=0, stat=0, threads=0, shared=False):
    mp.mp_set_int("many_cluster", cluster)
    mp.mp_set_int("many_stat", stat)
    mp.mp_set_int("many_threads", threads)
    M, N = pbs[0].psi32.shape
    P = len(pbs)
    if ld is None:
        ld = (N + 3) // 4 * 4
    if shared:
        buf = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")
        buf[:, :N] = dev(pbs[0].psi32)
        psi_d = buf[:, :N]
    else:
        buf = torch.full((P, M, ld), 7.0, dtype=torch.float32, device="cuda")      # pad columns hold garbage on purpose
        for q, pb in enumerate(pbs):
            buf[q, :, :N] = dev(pb.psi32)
        psi_d = buf[:, :, :N]
    Y = dev(np.stack([pb.Y[0] for pb in pbs]))
    res = mp.mp_recover_many(psi_d, Y, eps, max_iter, trace=True)
    torch.cuda.synchronize()
    return (res.x.cpu().numpy(), res.r.cpu().numpy(), res.n_iter.cpu().numpy(), res.idx_trace.cpu().numpy(), res.c_trace.cpu().numpy())


def grade_all(pbs, eps, max_iter, out, shared=False, **kw):
    X, R, T, I, Cc = out
    grades = []
    for q, pb in enumerate(pbs):
        t = int(T[q])
        psi = pbs[0].psi32 if shared else pb.psi32
        grades.append(grading.grade_single(psi, pb.Y[0], eps, max_iter, X[q], R[q], t, I[q, :t], Cc[q, :t], nthreads=4, **kw))
    return grades


SHAPES = [
    # N,    M,    K,  P, ld
    (256, 1024, 16, 5, None),     # cfg1's shape: 1 MiB per problem
    (250, 333, 8, 7, None),       # N % 4 != 0, odd atom counts per CTA
    (37, 50, 3, 20, 40),          # tiny: cluster size capped by the atom count, padded ld
    (1, 3, 1, 2, 4),              # N = 1
    (500, 1000, 20, 4, None),     # the paper's M = 1000 at rho = 0.5: 2 MB, stationary in a 16-CTA cluster
    (1000, 1000, 30, 3, None),    # rho = 1: 4 MB does not fit a cluster's shared memory -> streamed from L2
    (2048, 300, 12, 2, None),     # longest supported residual (V = 16)
    (130, 149, 6, 3, 256),        # ld > Npad
]


@pytest.mark.parametrize("N,M,K,P,ld", SHAPES)
def test_many_every_problem_graded_like_a_single_run(mp, N, M, K, P, ld):
    cfg, pbs = make_many(N, M, K, P, eps=1e-4, max_iter=6 * K + 3)
    out = run_many(mp, pbs, cfg.eps, cfg.max_iter, ld)
    assert mp.mp_get_int("info_many_cluster") >= 1
    grade_all(pbs, cfg.eps, cfg.max_iter, out)


@pytest.mark.parametrize("N,M,K,P", [(256, 1024, 16, 3), (250, 333, 8, 5), (600, 1000, 24, 3)])
def test_cluster_sizes_and_stationary_or_streamed_agree_bit_for_bit(mp, N, M, K, P):
    cfg, pbs = make_many(N, M, K, P, eps=1e-5, max_iter=8 * K)
    ref = run_many(mp, pbs, cfg.eps, cfg.max_iter)
    grade_all(pbs, cfg.eps, cfg.max_iter, ref)
    seen = set()
    for cluster in (1, 2, 4, 8, 16):
        for stat in (0, 2):
            for threads in (0, 64, 128):
                if threads and cluster not in (1, 8):
                    continue
                out = run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=cluster, stat=stat, threads=threads)
                seen.add((mp.mp_get_int("info_many_cluster"), mp.mp_get_int("info_many_stat")))
                assert _traces_equal(ref, out), f"cluster={cluster} stat={stat} threads={threads} differs from the auto plan"
    assert len(seen) >= 4                                                          # several cluster sizes, both modes ran


def _traces_equal(ref, out):
    """Everything but the unwritten tail of the traces (t >= n_iter) must be identical."""
    X, R, T, I, Cc = ref
    X2, R2, T2, I2, C2 = out
    if not (np.array_equal(X, X2) and np.array_equal(R, R2) and np.array_equal(T, T2)):
        return False
    return all(np.array_equal(I[q, :T[q]], I2[q, :T[q]]) and np.array_equal(Cc[q, :T[q]], C2[q, :T[q]]) for q in range(len(T)))


HARD_AT = [3, 29, 53, 79, 103]


def test_more_problems_than_clusters_and_mixed_stop_times(mp):
    """P far above the number of co-resident clusters (forced 16-CTA clusters: at most 9 on 148 SMs): clusters draw problems
    from the device counter; some problems stop at once (y = 0), some run to max_iter (sparsity beyond recovery)."""
    N, M, P = 64, 256, 120
    cfg, pbs = make_many(N, M, 3, P, eps=1e-5, max_iter=40)
    for q in range(0, P, 7):
        pbs[q].Y[0][:] = 0.0                                                       # 0 iterations
    _, hard = make_many(N, M, 40, 5, seed0=500, eps=1e-5, max_iter=40)             # K = 40 of N = 64: runs to max_iter
    for q, h in zip(HARD_AT, hard):
        pbs[q] = h
    out = run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=16)
    assert mp.mp_get_int("info_many_clusters") < P
    T = out[2]
    assert all(T[q] == 0 for q in range(0, P, 7)) and all(T[q] == 40 for q in HARD_AT)
    grade_all(pbs, cfg.eps, cfg.max_iter, out)
    out1 = run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=1)
    assert _traces_equal(out, out1)


def test_shared_dictionary_equals_single_signal_runs(mp):
    """problem_stride = 0: all problems share one dictionary -- each signal graded against the oracle on it, and
    bit-identical to the per-problem layout holding P copies."""
    N, M, K, P = 256, 1024, 12, 6
    cfg = problems.custom_config(N, M, K, B=P, eps=1e-5, max_iter=8 * K)
    pb = problems.make_problem(cfg, 3)
    pbs = [problems.Problem(cfg, pb.psi_raw, pb.psi32, pb.X[q:q + 1], pb.S[q:q + 1], pb.Y[q:q + 1]) for q in range(P)]
    out = run_many(mp, pbs, cfg.eps, cfg.max_iter, shared=True)
    grade_all(pbs, cfg.eps, cfg.max_iter, out, shared=True)
    out2 = run_many(mp, pbs, cfg.eps, cfg.max_iter, shared=False)
    assert _traces_equal(out, out2)


def test_edge_cases_many(mp):
    cfg, pbs = make_many(64, 200, 4, 3)
    M, N = pbs[0].psi32.shape
    X, R, T, _, _ = run_many(mp, pbs, 1e-5, 0)                                     # max_iter = 0 -> x = 0, r = y
    assert not T.any() and not X.any() and all(np.array_equal(R[q], pbs[q].Y[0]) for q in range(3))
    X, R, T, _, _ = run_many(mp, pbs, 1.0, 50)                                     # eps >= 1
    assert not T.any() and not X.any()
    out = run_many(mp, pbs, 0.0, 40)                                               # eps = 0 -> runs to max_iter
    assert (out[2] == 40).all()
    grade_all(pbs, 0.0, 40, out)
    out = run_many(mp, pbs, 0.0, 1)                                                # one gemv + argmax (Eq. 9, Eq. 16)
    for q in range(3):
        c_ref = oracle.correlate(pbs[q].psi32, pbs[q].Y[0].astype(np.float64))
        assert out[2][q] == 1 and out[3][q, 0] == oracle.argmax_abs(c_ref)


def test_tie_break_lowest_index_many(mp):
    """Duplicated and negated atoms placed in different CTAs of the cluster: the lowest index must win."""
    cfg, pbs = make_many(128, 512, 5, 2, eps=1e-5, max_iter=30)
    for pb in pbs:
        s = int(pb.S[0][np.argmax(np.abs(pb.X[0][pb.S[0]]))])                      # the first pick
        lo, hi = (s, 500) if s < 500 else (7, s)
        pb.psi32[hi] = pb.psi32[lo] if s == lo else -pb.psi32[s]
        if s != lo:
            pb.psi32[lo] = -pb.psi32[s]
    for cluster in (1, 16):
        out = run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=cluster)
        grade_all(pbs, cfg.eps, cfg.max_iter, out)
        for q, pb in enumerate(pbs):
            ref = oracle.mp(pb.psi32, pb.Y[0].astype(np.float64), float(np.float32(cfg.eps)), cfg.max_iter)
            assert out[3][q, 0] == ref.idx[0]


def test_phase_diagram_cell_paper_parameters(mp):
    """One cell of the paper's Fig. 1 experiment with its own parameters: M = 1000, Bernoulli +-1/sqrt(N)
    dictionaries (Eq. 13), K nonzeros from U[-1, 1], eps = 1e-7, T = N; rho = 0.5, sigma = 0.03 -- deep in the region
    where the paper reports exact recovery, so Eq. 14 must be ~0 for every trial, and every trial is fully graded."""
    M, N, K, P = 1000, 500, 30, 4
    cfg, pbs = make_many(N, M, K, P, seed0=40, dictionary="bernoulli", values="uniform", eps=1e-7, max_iter=N)
    out = run_many(mp, pbs, cfg.eps, cfg.max_iter)
    assert mp.mp_get_int("info_many_stat") == 1
    grade_all(pbs, cfg.eps, cfg.max_iter, out)
    for q, pb in enumerate(pbs):
        err = oracle.reconstruction_error_pct(out[0][q].astype(np.float64), pb.X[0])
        assert err < 1e-6, f"trial {q}: Eq. 14 error {err:.2e} %"


def test_long_residual_falls_back_to_single_signal_solves(mp):
    cfg, pbs = make_many(2100, 160, 5, 2, eps=1e-4, max_iter=30)
    out = run_many(mp, pbs, cfg.eps, cfg.max_iter)
    assert mp.mp_get_int("info_many_cluster") == 0
    grade_all(pbs, cfg.eps, cfg.max_iter, out)


def test_repeated_runs_are_bit_identical(mp):
    """Race detector of last resort (compute-sanitizer is not available on the pool): the exchange is st.async + mbarrier with
    alternating slots, the problems are drawn from a device counter -- 25 runs of a 150-problem batch, in three plans, must give
    the same bits every time (a lost or stale key, or a slot overwritten too early, shows up as a different trace)."""
    cfg, pbs = make_many(96, 400, 6, 150, eps=1e-5, max_iter=40)
    for cluster, stat in ((0, 0), (16, 0), (4, 2)):
        ref = run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=cluster, stat=stat)
        for _ in range(24):
            assert _traces_equal(ref, run_many(mp, pbs, cfg.eps, cfg.max_iter, cluster=cluster, stat=stat))
    grade_all(pbs[:20], cfg.eps, cfg.max_iter, tuple(a[:20] for a in ref))


def test_random_shapes_against_the_oracle(mp):
    """A fixed-seed sweep over awkward shapes (N around the 128-float register classes, tiny and odd M, NaN in the pad columns
    of the dictionary), three plans each: every problem fully graded."""
    rng = np.random.default_rng(123)
    for trial in range(14):
        N = int(rng.choice([1, 3, 31, 33, 127, 129, 257, 385, 500, 641, 777, 1025, 1281, 1793, 2047]))
        M = int(rng.choice([1, 2, 15, 17, 33, 100, 255, 300, 1000]))
        if 4 * N * M > 4e6:
            M = max(1, int(4e6 / (4 * N)))
        K = max(1, min(M, N // 6 + 1, 10))
        P = int(rng.choice([1, 3, 9]))
        cfg = problems.custom_config(N, M, K, dictionary="bernoulli" if trial % 3 == 0 else "gaussian", eps=1e-5, max_iter=4 * K + 2)
        pbs = [problems.make_problem(cfg, 2000 + 7 * trial + q) for q in range(P)]
        ld = (N + 3) // 4 * 4 + 4 * (trial % 2)
        buf = torch.full((P, M, ld), float("nan"), dtype=torch.float32, device="cuda")
        for q, pb in enumerate(pbs):
            buf[q, :, :N] = dev(pb.psi32)
        Y = dev(np.stack([pb.Y[0] for pb in pbs]))
        for knobs in ({}, {"many_stat": 2}, {"many_cluster": int(rng.choice([1, 2, 4, 8, 16]))}):
            for k in ("many_stat", "many_cluster", "many_threads"):
                mp.mp_set_int(k, knobs.get(k, 0))
            res = mp.mp_recover_many(buf[:, :, :N], Y, cfg.eps, cfg.max_iter, trace=True)
            torch.cuda.synchronize()
            out = tuple(a.cpu().numpy() for a in (res.x, res.r, res.n_iter, res.idx_trace, res.c_trace))
            grade_all(pbs, cfg.eps, cfg.max_iter, out)
