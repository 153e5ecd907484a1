"""GPU parity tests: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle on the
same seeded inputs.  Contract and readings: tests/grading.py and DESIGN.md.  Run on a B200: pytest -m gpu.
"""
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
    m.mp_set_int("algo", 0)
    m.mp_set_int("batched_algo", 0)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_single(mp, psi32, y32, eps, max_iter, algo=0, ld=None):
    """-> (x, r, n_iter, idx, c) as numpy"""
    mp.mp_set_int("algo", algo)
    M, N = psi32.shape
    if ld is None:
        ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")     # pad columns hold garbage on purpose
    buf[:, :N] = dev(psi32)
    psi_d = buf[:, :N]
    res = mp.mp_recover(psi_d, dev(y32), eps, max_iter, trace=True)
    torch.cuda.synchronize()
    t = int(res.n_iter.item())
    return (res.x.cpu().numpy(), res.r.cpu().numpy(), t, res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t])


ALGOS = [1, 2, 3, 4]   # 1 = TMA-staged persistent kernel, 2 = stream loop, 3 = register-streaming persistent kernel,
                       # 4 = one thread-block cluster (the mp_recover_many kernel with P = 1; N <= 2048)


# ------------------------------------------------------------------------------------------ normalisation (a0)
@pytest.mark.parametrize("N,M", [(256, 1024), (250, 33), (1, 5), (4096, 300), (37, 1000)])
def test_normalize_columns_matches_float64_quotient(mp, N, M):
    """Eq. 4: fp32 result == float64 normalise-then-round, to <= 1 ulp; ||psi_m|| = 1 to 2e-7."""
    raw = synth.gaussian_dictionary(N, M, seed=11)
    raw[M // 2] = 0.0                                                       # a zero atom stays zero (reading R7)
    ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 3.0, dtype=torch.float32, device="cuda")
    buf[:, :N] = dev(raw)
    norms = torch.empty(M, dtype=torch.float32, device="cuda")
    mp.mp_normalize_columns(buf[:, :N], norms)
    torch.cuda.synchronize()
    got = buf[:, :N].cpu().numpy()
    ref64, n64 = oracle.normalize_columns(raw)
    ref = ref64.astype(np.float32)
    ulp = np.spacing(np.abs(ref)).astype(np.float64)
    assert np.all(np.abs(got.astype(np.float64) - ref.astype(np.float64)) <= ulp)
    assert np.array_equal(got, ref) or np.mean(got != ref) < 1e-3           # float64 quotient rounded once: essentially always equal
    np.testing.assert_allclose(norms.cpu().numpy(), n64, rtol=1e-6)
    nn = np.linalg.norm(got.astype(np.float64), axis=1)
    keep = np.arange(M) != M // 2
    assert np.all(np.abs(nn[keep] - 1.0) <= 2e-7) and nn[M // 2] == 0.0
    if ld > N:
        assert torch.all(buf[:, N:] == 3.0)                                  # pad columns untouched


def test_normalize_leaves_unit_bernoulli_unchanged(mp):
    """Eq. 13: +-1/sqrt(N) atoms are unit already; with N a power of 4 the kernel returns them bit-identical."""
    raw = synth.bernoulli_dictionary(1024, 200, seed=5)
    d = dev(raw)
    mp.mp_normalize_columns(d)
    assert np.array_equal(d.cpu().numpy(), raw)


# ------------------------------------------------------------------------------------------ CFG1, all seeds, both algorithms
@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_cfg1_full_grading(mp, seed, algo):
    pb = problems.make_problem(synth.config("cfg1"), seed)
    c = pb.cfg
    x, r, t, idx, cc = run_single(mp, pb.psi32, pb.Y[0], c.eps, c.max_iter, algo)
    g = grading.grade_single(pb.psi32, pb.Y[0], c.eps, c.max_iter, x, r, t, idx, cc, x_true=pb.X[0], support=pb.S[0])
    assert g.exact_recovery
    assert g.first_divergence >= 0 or g.n_iter_gpu == g.n_iter_ref or abs(g.n_iter_gpu - g.n_iter_ref) == 1


# ------------------------------------------------------------------------------------------ ragged shapes / several tiles + tail
RAGGED = [
    # N,    M,    K,  ld     what it exercises
    (250, 1000, 10, None),   # N % 4 != 0 (pad columns in ld), M not a multiple of anything
    (37, 5, 2, 40),          # fewer atoms than CTAs, tiny N
    (1, 3, 1, 4),            # N = 1
    (130, 149, 6, 256),      # ld > Npad (non-contiguous atoms), M = grid + 1
    (2052, 777, 20, None),   # N just above a 128 multiple
    (5000, 600, 24, None),   # row > one pipeline slot: column-chunked path
    (8192, 320, 16, None),   # largest N of the configs
    (512, 4099, 24, None),   # many atoms per CTA, ragged tail
]


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("N,M,K,ld", RAGGED)
def test_ragged_shapes_full_grading(mp, N, M, K, ld, algo):
    if algo == 4 and N > 2048:
        pytest.skip("the cluster kernel holds the residual in registers: N <= 2048")
    cfg = problems.custom_config(N, M, K, eps=1e-4, max_iter=6 * K + 3)
    pb = problems.make_problem(cfg, seed=4)
    x, r, t, idx, cc = run_single(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, algo, ld)
    grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, x, r, t, idx, cc)


@pytest.mark.parametrize("f64", [False, True])
@pytest.mark.parametrize("N,M,K,ld", RAGGED + [(64, 5000, 8, None), (200, 3000, 8, None), (500, 2000, 8, None), (1500, 40000, 12, None)])
def test_forced_l2_plan_on_ragged_shapes(mp, N, M, K, ld, f64):
    """The L2 mechanisms of the register-streaming kernels (reversed order on odd iterations, pinned rows kept off the ends of a share,
    items drawn from a counter when the shares are long) only engage by themselves above 90 MB.  Here they are forced onto small ragged
    shapes -- every (A, UC) variant, shares of 0, 1 and a few groups, a few pinned rows per share -- and must leave every output
    bit unchanged against the run with all of them off; the forced run is graded in full."""
    cfg = problems.custom_config(N, M, K, eps=1e-4, max_iter=6 * K + 3)
    pb = problems.make_problem(cfg, seed=5)

    def run():
        if not f64:
            return run_single(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, 3, ld)
        ld2 = ((ld or N) + 1) // 2 * 2
        psi = torch.zeros(M, ld2, dtype=torch.float64, device="cuda")[:, :N]; psi.copy_(torch.from_numpy(pb.psi32.astype(np.float64)))
        res = mp.mp_recover_f64(psi, torch.from_numpy(pb.Y[0].astype(np.float64)).cuda(), cfg.eps, cfg.max_iter, trace=True)
        torch.cuda.synchronize()
        t = int(res.n_iter.item())
        return (res.x.cpu().numpy(), res.r.cpu().numpy(), t, res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t])

    mp.mp_set_int("pingpong", 1); mp.mp_set_int("l2_resident_mb", 1); mp.mp_set_int("balance", 1)
    try:
        off = run()
        for mb in (1, 2, 5):                                                     # no pinned rows / 2 MB / 5 MB of them (if the dictionary is larger)
            mp.mp_set_int("pingpong", 2); mp.mp_set_int("l2_resident_mb", mb); mp.mp_set_int("balance", 0)
            on = run()
            for a, b in zip(off, on):
                assert np.array_equal(a, b)
    finally:
        mp.mp_set_int("pingpong", 0); mp.mp_set_int("l2_resident_mb", 0); mp.mp_set_int("balance", 0)
    if not f64:
        x, r, t, idx, cc = on
        grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, x, r, t, idx, cc)


@pytest.mark.parametrize("N,M,K", [(20000, 64, 8), (16, 200000, 4), (19000, 160, 6), (3, 100000, 1)])
def test_extreme_aspect_ratios_auto_dispatch(mp, N, M, K):
    """Shapes at the edges of the kernels' plans under algo = auto: a residual too long for shared memory (stream loop),
    a very long residual that still fits, and very many very short atoms."""
    cfg = problems.custom_config(N, M, K, eps=1e-4, max_iter=4 * K + 2)
    pb = problems.make_problem(cfg, seed=8)
    x, r, t, idx, cc = run_single(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, 0)
    grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, x, r, t, idx, cc)
    assert mp.mp_get_int("info_algo") == (2 if N == 20000 else 3)


# ------------------------------------------------------------------------------------------ edge / degenerate cases
@pytest.mark.parametrize("algo", ALGOS)
def test_edge_cases(mp, algo):
    pb = problems.make_problem(problems.custom_config(64, 200, 4), seed=2)
    y = pb.Y[0]
    # y = 0 -> 0 iterations (0 > eps*0 is false)
    x, r, t, _, _ = run_single(mp, pb.psi32, np.zeros_like(y), 1e-5, 50, algo)
    assert t == 0 and not x.any() and not r.any()
    # max_iter = 0 -> x = 0, r = y
    x, r, t, _, _ = run_single(mp, pb.psi32, y, 1e-5, 0, algo)
    assert t == 0 and not x.any() and np.array_equal(r, y)
    # eps >= 1 -> ||y|| > eps ||y|| is false
    x, r, t, _, _ = run_single(mp, pb.psi32, y, 1.0, 50, algo)
    assert t == 0 and np.array_equal(r, y)
    # eps = 0 -> runs to max_iter (no exact zero residual on random data)
    x, r, t, idx, cc = run_single(mp, pb.psi32, y, 0.0, 40, algo)
    assert t == 40
    grading.grade_single(pb.psi32, y, 0.0, 40, x, r, t, idx, cc)
    # max_iter = 1: one gemv + argmax (Eq. 9, Eq. 16)
    x, r, t, idx, cc = run_single(mp, pb.psi32, y, 0.0, 1, algo)
    c_ref = oracle.correlate(pb.psi32, y.astype(np.float64))
    assert t == 1 and idx[0] == oracle.argmax_abs(c_ref) and abs(cc[0] - c_ref[idx[0]]) <= 1e-6 * np.linalg.norm(y)


@pytest.mark.parametrize("algo", ALGOS)
def test_orthonormal_hadamard_recovers_in_k_steps(mp, algo):
    """north_star pin on the GPU path: Psi = Hadamard/sqrt(N), N = M = 256 (entries +-1/16 exact): K steps, x~ = x."""
    n = 256
    H = np.array([[1.0]])
    while H.shape[0] < n:
        H = np.block([[H, H], [H, -H]])
    psi32 = np.ascontiguousarray((H / 16.0).T.astype(np.float32))
    x_true = np.zeros(n)
    S = [3, 77, 200, 129, 255, 0]
    x_true[S] = [2.0, -1.5, 0.75, 3.25, -0.5, 1.0]                          # exactly representable, distinct magnitudes
    y = (H / 16.0) @ x_true
    x, r, t, idx, cc = run_single(mp, psi32, y.astype(np.float32), 1e-6, 100, algo)
    order = [S[k] for k in np.argsort(-np.abs(x_true[S]), kind="stable")]
    assert t == len(S) and list(idx) == order
    np.testing.assert_allclose(x, x_true, atol=1e-6)
    assert np.linalg.norm(r) <= 1e-6 * np.linalg.norm(y)


@pytest.mark.parametrize("algo", ALGOS)
def test_tie_break_lowest_index(mp, algo):
    """Eq. 16: duplicated and negated atoms have exactly equal |c|; the smaller index must win,
    wherever the two copies fall (same warp, different warps, different CTAs)."""
    pb = problems.make_problem(problems.custom_config(128, 600, 4), seed=9)
    psi = pb.psi32.copy()
    y = pb.Y[0]
    c = oracle.correlate(psi, y.astype(np.float64))
    best = int(oracle.argmax_abs(c))
    for other, sign in [(best + 1 if best + 1 < 600 else best - 1, 1.0), (599 - best if 599 - best != best else 0, -1.0), (0 if best else 1, 1.0)]:
        p = psi.copy()
        p[other] = sign * p[best]
        x, r, t, idx, cc = run_single(mp, p, y, 0.0, 1, algo)
        assert idx[0] == min(best, other), (best, other, idx[0])
        assert np.sign(cc[0]) == (np.sign(c[best]) if idx[0] == best else sign * np.sign(c[best]))
    # all |c| equal: Hadamard/sqrt(N) with y = e_0 -> index 0
    n = 64
    H = np.array([[1.0]])
    while H.shape[0] < n:
        H = np.block([[H, H], [H, -H]])
    e0 = np.zeros(n, np.float32); e0[0] = 1.0
    x, r, t, idx, cc = run_single(mp, np.ascontiguousarray((H / 8.0).T.astype(np.float32)), e0, 0.0, 1, algo)
    assert idx[0] == 0 and cc[0] == 0.125


def test_rerun_is_bit_identical_and_workspace_reusable(mp):
    """Deterministic reduction order: two runs give identical bits; a dirty workspace does not matter."""
    pb = problems.make_problem(synth.config("cfg1"), 2)
    mp.mp_set_int("algo", 0)
    psi_d, y_d = dev(pb.psi32), dev(pb.Y[0])
    ws = torch.empty(mp.mp_workspace_bytes(256, 1024, 1) + 256, dtype=torch.uint8, device="cuda").fill_(0xAB)
    a = mp.mp_recover(psi_d, y_d, 1e-5, 4096, trace=True, workspace=ws)
    torch.cuda.synchronize()
    xa, ra, ta = a.x.clone(), a.r.clone(), int(a.n_iter.item())
    ia = a.idx_trace[:ta].clone()
    b = mp.mp_recover(psi_d, y_d, 1e-5, 4096, trace=True, workspace=ws)
    torch.cuda.synchronize()
    assert int(b.n_iter.item()) == ta and torch.equal(b.x, xa) and torch.equal(b.r, ra) and torch.equal(b.idx_trace[:ta], ia)


def test_invalid_arguments_on_device(mp):
    pb = problems.make_problem(problems.custom_config(64, 100, 3), seed=1)
    psi_d, y_d = dev(pb.psi32), dev(pb.Y[0])
    with pytest.raises(mp.MPError) as e:
        mp.mp_recover(psi_d, y_d, -1.0, 10)
    assert e.value.status == mp.MP_ERR_INVALID_ARG
    with pytest.raises(mp.MPError) as e:
        mp.mp_recover(psi_d, y_d, 1e-5, 10, workspace=torch.empty(300, dtype=torch.uint8, device="cuda"))
    assert e.value.status == mp.MP_ERR_WORKSPACE


# ------------------------------------------------------------------------------------------ CFG2 (full replay) and CFG3 (sampled)
def test_cfg2_full_grading(mp):
    pb = problems.make_problem(synth.config("cfg2"), 1)
    c = pb.cfg
    x, r, t, idx, cc = run_single(mp, pb.psi32, pb.Y[0], c.eps, c.max_iter, 0)
    g = grading.grade_single(pb.psi32, pb.Y[0], c.eps, c.max_iter, x, r, t, idx, cc, x_true=pb.X[0], support=pb.S[0])
    assert g.exact_recovery and 500 < g.n_iter_gpu < 1200


def test_cfg3_full_size_sampled_grading(mp):
    """Fast pre-check (the every-iteration grading of cfg3, seeds 1-3, is tests/test_gpu_fullsize.py).
    BASELINE.json's headline size (N=4096, M=16384, 256 MiB Psi) in the launch configuration bench.py times:
    every 97th iteration plus the first/last few are rebuilt in float64 from the GPU trace and checked one by one;
    properties that hold at any size (monotone norm via the trace, stop rule, support) are checked on all."""
    pb = problems.make_problem(synth.config("cfg3"), 1)
    c = pb.cfg
    x, r, t, idx, cc = run_single(mp, pb.psi32, pb.Y[0], c.eps, c.max_iter, 0)
    assert 800 < t < 2500
    ts = sorted(set(list(range(0, 4)) + list(range(5, t, 97)) + list(range(t - 3, t))))
    grading.grade_sampled(pb.psi32, pb.Y[0], idx, cc, t, r, ts)
    # support: MP at N = 16K never picks an off-support atom -> selected atoms == true support
    assert set(idx.tolist()) == set(pb.S[0].tolist())
    coef = np.zeros(c.M); np.add.at(coef, idx, cc.astype(np.float64))
    assert np.all(np.abs(x - coef) <= 6e-8 * np.abs(coef) + 1e-45)
    assert np.linalg.norm(x - pb.X[0]) <= 1e-4 * np.linalg.norm(pb.X[0])
    ny = np.linalg.norm(pb.Y[0].astype(np.float64))
    assert np.linalg.norm(r.astype(np.float64)) <= np.float32(c.eps) * ny * (1 + 1e-6)


# ------------------------------------------------------------------------------------------ batched (a9)
BATCHED_ALGOS = [1, 2, 3]     # 1 = lock-step tensor-core kernel (split-TF32 tcgen05), 2 = sequential single-signal solves,
                              # 3 = one thread-block cluster per signal on the shared dictionary


@pytest.mark.parametrize("B,N,M", [(64, 2048, 8192), (7, 250, 333), (64, 128, 512), (1, 4096, 2048), (33, 1000, 9000)])
def test_batched_correlation_matches_float64_oracle(mp, B, N, M):
    """The contraction of the batched path alone: C = Psi^T Y on the tensor cores against the oracle's float64
    ascending-n dot products (Eq. 9), every element, tolerance C_TOL * ||y_b||."""
    cfg = problems.custom_config(N, M, max(1, N // 16), B=B)
    psi32 = problems.normalise_on_host(synth.make_dictionary(cfg, seed=11))
    rng = np.random.default_rng(5)
    Y = rng.standard_normal((B, N)).astype(np.float32)
    Y[:, ::7] *= 1e-3                                                        # mixed magnitudes inside one residual
    ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 3.0, dtype=torch.float32, device="cuda"); buf[:, :N] = dev(psi32)
    Yb = torch.full((B, ld), -2.0, dtype=torch.float32, device="cuda"); Yb[:, :N] = dev(Y)
    Cg = mp.mp_correlate_batched(buf[:, :N], Yb[:, :N])
    torch.cuda.synchronize()
    Cg = Cg.cpu().numpy().astype(np.float64)
    worst = 0.0
    for b in range(B):
        ref = oracle.correlate(psi32, Y[b].astype(np.float64), nthreads=oracle.default_threads())
        err = np.abs(Cg[b] - ref).max() / np.linalg.norm(Y[b].astype(np.float64))
        worst = max(worst, err)
    assert worst <= grading.C_TOL, worst


@pytest.mark.parametrize("algo", BATCHED_ALGOS)
@pytest.mark.parametrize("B,N,M,K", [(3, 256, 1024, 16), (5, 250, 333, 8), (64, 128, 512, 6), (9, 512, 9000, 24)])
def test_batched_every_signal_graded_like_a_single_run(mp, B, N, M, K, algo):
    """P:165 / reading R17: signal b's result is MP on (Psi, y_b) under the same rules as the single-signal path
    (full teacher-forced grading per signal through the traced entry point); finished signals are frozen."""
    cfg = problems.custom_config(N, M, K, eps=1e-5, max_iter=10 * K, B=B)
    pb = problems.make_problem(cfg, seed=6)
    pb.Y[B // 2] = 0.0                                                       # one signal that stops at once
    mp.mp_set_int("batched_algo", algo)
    ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 5.0, dtype=torch.float32, device="cuda"); buf[:, :N] = dev(pb.psi32)
    Yb = torch.full((B, ld), 9.0, dtype=torch.float32, device="cuda"); Yb[:, :N] = dev(pb.Y)
    res = mp.mp_recover_batched(buf[:, :N], Yb[:, :N], cfg.eps, cfg.max_iter, trace=True)
    torch.cuda.synchronize()
    X, R, T = res.x.cpu().numpy(), res.r.cpu().numpy(), res.n_iter.cpu().numpy()
    I, Cc = res.idx_trace.cpu().numpy(), res.c_trace.cpu().numpy()
    assert T[B // 2] == 0 and not X[B // 2].any() and not R[B // 2].any()
    c_tol = grading.c_tol_tensor_core(N) if algo == 1 else grading.C_TOL
    for b in range(B):
        t = int(T[b])
        grading.grade_single(pb.psi32, pb.Y[b], cfg.eps, cfg.max_iter, X[b], R[b], t, I[b, :t], Cc[b, :t],
                             x_true=pb.X[b], support=pb.S[b], nthreads=1, c_tol=c_tol)
    # and the untraced entry point gives the same bits
    res2 = mp.mp_recover_batched(buf[:, :N], Yb[:, :N], cfg.eps, cfg.max_iter)
    torch.cuda.synchronize()
    assert torch.equal(res2.x, res.x) and torch.equal(res2.r, res.r) and torch.equal(res2.n_iter, res.n_iter)


# ------------------------------------------------------------------------------------------ encode + score on device (NEXT 1)
@pytest.mark.parametrize("N,M,K", [(256, 1024, 16), (250, 333, 8), (4096, 16384, 256), (37, 1000, 700), (2048, 8192, 0)])
def test_encode_sparse_is_bit_exact(mp, N, M, K):
    """Eq. 2: the device encode equals the oracle's ascending-k float64 sum rounded to fp32 once, bit for bit (the
    products double(float)*double(float) are exact, the adds run in the same order)."""
    cfg = problems.custom_config(N, M, max(K, 1))
    psi32 = problems.normalise_on_host(synth.make_dictionary(cfg, seed=4))
    rng = np.random.default_rng(9)
    idx = rng.integers(0, M, K).astype(np.int32)                             # with replacement: repeats accumulate
    val = rng.standard_normal(K).astype(np.float32)
    ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 3.0, dtype=torch.float32, device="cuda"); buf[:, :N] = dev(psi32)
    y = mp.mp_encode_sparse(buf[:, :N], dev(idx), dev(val))
    torch.cuda.synchronize()
    ref = oracle.encode_sparse(psi32, idx, val.astype(np.float64)).astype(np.float32)
    assert np.array_equal(y.cpu().numpy(), ref)
    if K:                                                                    # an out-of-range index contributes nothing
        bad = idx.copy(); bad[0] = M + 5
        y2 = mp.mp_encode_sparse(buf[:, :N], dev(bad), dev(val)).cpu().numpy()
        ref2 = oracle.encode_sparse(psi32, idx[1:], val[1:].astype(np.float64)).astype(np.float32)
        assert np.array_equal(y2, ref2)


def test_encode_recover_score_pipeline_on_device(mp):
    """encode -> mp_recover -> score without host data (CFG1): the recovered x~ scores Eq. 14 like the oracle's
    formula on the same vectors, and the error is at the "recovers exactly" level."""
    pb = problems.make_problem(synth.config("cfg1"), 2)
    c = pb.cfg
    psi_d = dev(pb.psi32)
    order = np.sort(pb.S[0])
    y_d = mp.mp_encode_sparse(psi_d, dev(order.astype(np.int32)), dev(pb.X[0][order].astype(np.float32)))
    x32 = pb.X[0][order].astype(np.float32)                                  # the device encode takes fp32 coefficients
    assert np.array_equal(y_d.cpu().numpy(), oracle.encode_sparse(pb.psi32, order, x32.astype(np.float64)).astype(np.float32))
    res = mp.mp_recover(psi_d, y_d, c.eps, c.max_iter)
    x_true_d = dev(pb.X[0].astype(np.float32))
    e = mp.mp_reconstruction_error(res.x, x_true_d)
    torch.cuda.synchronize()
    ref = oracle.reconstruction_error_pct(res.x.cpu().numpy().astype(np.float64), pb.X[0].astype(np.float32).astype(np.float64))
    assert abs(e.item() - ref) <= 1e-12 * ref and e.item() < 1e-6
    # a hand-computed case: (0.1^2 + 0.1^2) / 1 * 100 = 2 %
    e2 = mp.mp_reconstruction_error(dev(np.array([0.9, 0.1, 0.0], np.float32)), dev(np.array([1.0, 0.0, 0.0], np.float32)))
    assert abs(e2.item() - 2.0) < 1e-5


# ------------------------------------------------------------------------------------------ host-buffer entry points (e2e path)
def test_host_entry_point_matches_device_entry_point(mp):
    pb = problems.make_problem(synth.config("cfg1"), 3)
    mp.mp_set_int("algo", 0)
    h = mp.mp_recover_host(torch.from_numpy(pb.psi_raw), torch.from_numpy(pb.Y[0]), 1e-5, 4096, normalize=True, trace=True)
    t = int(h.n_iter.item())
    x, r, t2, idx, cc = run_single(mp, pb.psi32, pb.Y[0], 1e-5, 4096, 0)
    assert t == t2 and np.array_equal(h.idx_trace.numpy()[:t], idx)
    assert np.array_equal(h.x.numpy(), x) and np.array_equal(h.r.numpy(), r)


def test_dictionary_handle_matches_the_other_entry_points_bit_for_bit(mp):
    """P:165 "the host to device dictionary transfer only takes place once": a handle created from HOST memory (chunked
    upload + normalisation on the device) and one that borrows a DEVICE tensor give, call after call, exactly the bits of
    mp_recover_host / mp_recover / mp_recover_batched; several signals through one handle; traces; raw C-ABI use."""
    import ctypes as C
    pb = problems.make_problem(problems.custom_config(250, 3000, 12, eps=1e-5, max_iter=96, B=5), seed=3)
    raw_odd = torch.from_numpy(pb.psi_raw)                                     # host row stride 250: not a multiple of 4
    raw = torch.zeros(3000, 252); raw[:, :250] = raw_odd; raw = raw[:, :250]   # the same dictionary with a padded stride
    hh = mp.mp_dictionary_create(raw_odd, normalize=True)                      # host -> device (re-pitched), normalised there
    psi_d = torch.zeros(3000, 252, device="cuda")[:, :250]; psi_d.copy_(raw_odd)   # device row stride 252 (the boundary wants ld % 4 == 0)
    mp.mp_normalize_columns(psi_d); torch.cuda.synchronize()
    assert hh.N == 250 and hh.M == 3000 and hh.psi_ptr != 0
    hd = mp.mp_dictionary_create(psi_d)                                        # borrowed device tensor
    assert hd.psi_ptr == psi_d.data_ptr()
    for b in range(3):
        y = torch.from_numpy(pb.Y[b])
        ref = mp.mp_recover_host(raw, y, 1e-5, 96, normalize=True, trace=True)
        t = int(ref.n_iter.item())
        for h in (hh, hd):
            got = mp.mp_recover_host_h(h, y, 1e-5, 96, trace=True)
            assert int(got.n_iter.item()) == t and torch.equal(got.x, ref.x) and torch.equal(got.r, ref.r)
            assert torch.equal(got.idx_trace[:t], ref.idx_trace[:t]) and torch.equal(got.c_trace[:t], ref.c_trace[:t])
    grading.grade_single(psi_d.cpu().contiguous().numpy(), pb.Y[2], 1e-5, 96, got.x.numpy(), got.r.numpy(), t, got.idx_trace.numpy()[:t], got.c_trace.numpy()[:t])
    # batched through the handle == mp_recover_batched on device tensors
    Y_d = torch.zeros(5, 252, device="cuda")[:, :250]; Y_d.copy_(torch.from_numpy(pb.Y))      # the boundary wants ldy % 4 == 0
    refb = mp.mp_recover_batched(psi_d, Y_d, 1e-5, 96, trace=True)
    torch.cuda.synchronize()
    gotb = mp.mp_recover_batched_host_h(hh, torch.from_numpy(pb.Y), 1e-5, 96, trace=True)
    assert torch.equal(gotb.x, refb.x.cpu()) and torch.equal(gotb.r, refb.r.cpu()) and torch.equal(gotb.n_iter, refb.n_iter.cpu())
    for b in range(5):
        tb = int(gotb.n_iter[b])
        assert torch.equal(gotb.idx_trace[b, :tb], refb.idx_trace[b, :tb].cpu())
    # the C ABI raw: info returns shape and device pointer; a second create / destroy cycle leaves nothing behind
    N, M, ld, p = C.c_int(), C.c_int(), C.c_int64(), C.c_void_p()
    assert mp.binding.lib.mp_dictionary_info(hh.ptr, C.byref(N), C.byref(M), C.byref(ld), C.byref(p)) == 0
    assert (N.value, M.value, ld.value) == (250, 3000, 252) and p.value == hh.psi_ptr
    mp.mp_dictionary_destroy(hh); mp.mp_dictionary_destroy(hd); mp.mp_dictionary_destroy(hd)          # idempotent
    assert hh.ptr == 0


def test_automatic_l2_plan_by_dictionary_size(mp):
    """The plan the register-streaming kernel reports for itself (mp_internal.h l2_plan): same order and no pinned rows while the
    dictionary fits the L2, reversed order alone for 90-140 MB, reversed order + 88 MB of pinned rows above; whatever the plan, the
    outputs are the same bits as with everything switched off."""
    for N, M, want_pp, want_mb in ((2048, 8192, 0, 0), (2048, 14336, 1, 0), (2048, 22528, 1, 88)):
        g = torch.Generator(device="cuda"); g.manual_seed(N + M)
        psi = torch.randn(M, N, device="cuda", generator=g); mp.mp_normalize_columns(psi)
        y = torch.randn(N, device="cuda", generator=g)
        mp.mp_set_int("algo", 3)
        a = mp.mp_recover(psi, y, 0.0, 24, trace=True); torch.cuda.synchronize()
        assert mp.mp_get_int("info_l2_pingpong") == want_pp
        assert abs(mp.mp_get_int("info_l2_resident_mb") - want_mb) <= 6
        mp.mp_set_int("pingpong", 1); mp.mp_set_int("l2_resident_mb", 1); mp.mp_set_int("balance", 1)
        try:
            b = mp.mp_recover(psi, y, 0.0, 24, trace=True); torch.cuda.synchronize()
            assert mp.mp_get_int("info_l2_pingpong") == 0 and mp.mp_get_int("info_l2_resident_mb") == 0
        finally:
            mp.mp_set_int("pingpong", 0); mp.mp_set_int("l2_resident_mb", 0); mp.mp_set_int("balance", 0); mp.mp_set_int("algo", 0)
        assert torch.equal(a.x, b.x) and torch.equal(a.r, b.r) and torch.equal(a.idx_trace, b.idx_trace) and torch.equal(a.c_trace, b.c_trace)
        del psi


# ------------------------------------------------------------------------------------------ the paper's row-major layout
@pytest.mark.parametrize("aligned", [False, True])
@pytest.mark.parametrize("N,M,ldr", [(256, 1024, None), (250, 333, 340), (1, 5, None), (4096, 300, None), (37, 1000, 1003), (65, 129, None),
                                     (130, 250, 252), (63, 67, 68)])
def test_rowmajor_ingestion_is_bit_exact(mp, N, M, ldr, aligned):
    """mp_transpose_rowmajor against the oracle's element-by-element definition (A2 P:360 layout -> atom-major): bit-exact,
    pad columns of the destination untouched, odd source strides and unaligned source pointers accepted."""
    rng = np.random.default_rng(N * 1000 + M)
    psi = rng.standard_normal((N, M)).astype(np.float32)
    ldr = ldr or M
    off = 0 if aligned else 1                                                      # 16-byte aligned (128-bit kernel if ldr % 4 == 0) or not
    src = torch.full((N * ldr + 1,), -3.0, dtype=torch.float32, device="cuda")
    src_v = src[off:off + N * ldr].view(N, ldr)[:, :M]
    src_v.copy_(dev(psi))
    ld = (N + 3) // 4 * 4 + 4
    dst = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda")
    out = mp.mp_transpose_rowmajor(src_v, dst[:, :N])
    torch.cuda.synchronize()
    want = oracle.atom_major_from_rowmajor(psi)
    assert np.array_equal(out.cpu().numpy(), want)
    assert (dst[:, N:] == 7.0).all()


def test_solve_from_the_papers_layout(mp):
    """Row-major Bernoulli dictionary as the paper's program builds it -> transpose -> mp_recover: full grading."""
    pb = problems.make_problem(synth.config("cfg1"), 2)
    rowmajor = np.ascontiguousarray(pb.psi32.T)                                    # psi[n*M + m]
    psi_t = mp.mp_transpose_rowmajor(dev(rowmajor))
    c = pb.cfg
    res = mp.mp_recover(psi_t, dev(pb.Y[0]), c.eps, c.max_iter, trace=True)
    torch.cuda.synchronize()
    t = int(res.n_iter.item())
    g = grading.grade_single(pb.psi32, pb.Y[0], c.eps, c.max_iter, res.x.cpu().numpy(), res.r.cpu().numpy(), t,
                             res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t], x_true=pb.X[0], support=pb.S[0])
    assert g.exact_recovery


@pytest.mark.parametrize("N,M,K", [(1002, 19000, 40), (300, 64000, 24)])
def test_l2_residency_hints_do_not_change_results(mp, N, M, K):
    """The L2::evict_last / evict_first loads of the register-streaming kernel (auto for dictionaries above 110 MB; forced here
    on 76 MB ones with the knob): ragged N, full grading, and bit-identical results with the hints switched off."""
    cfg = problems.custom_config(N, M, K, eps=1e-5, max_iter=6 * K)
    pb = problems.make_problem(cfg, seed=9)
    mp.mp_set_int("l2_resident_mb", 40)
    try:
        out = run_single(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, 3)
        grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, *out, x_true=pb.X[0], support=pb.S[0])
        mp.mp_set_int("l2_resident_mb", 1)
        off = run_single(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, 3)
    finally:
        mp.mp_set_int("l2_resident_mb", 0)
    for a, b in zip(out, off):
        assert np.array_equal(a, b)


def test_l2_plan_scales_with_the_l2_size(mp):
    """The plan's thresholds are fractions of cudaDevAttrL2CacheSize (mp_internal.h l2_scale): with the attribute overridden to a
    quarter of this device's L2 through the knob "l2_bytes", a 64 MiB dictionary -- which the real L2 simply holds -- gets what a
    256 MiB one gets by default (reversed order, a quarter of 88 MB pinned), and the outputs are still the same bits."""
    N, M = 2048, 8192
    g = torch.Generator(device="cuda"); g.manual_seed(77)
    psi = torch.randn(M, N, device="cuda", generator=g); mp.mp_normalize_columns(psi)
    y = torch.randn(N, device="cuda", generator=g)
    mp.mp_set_int("algo", 3)
    try:
        a = mp.mp_recover(psi, y, 0.0, 24, trace=True); torch.cuda.synchronize()
        real = mp.mp_get_int("info_l2_bytes")
        assert real == torch.cuda.get_device_properties(0).L2_cache_size
        assert mp.mp_get_int("info_l2_pingpong") == 0 and mp.mp_get_int("info_l2_resident_mb") == 0
        mp.mp_set_int("l2_bytes", real // 4)
        b = mp.mp_recover(psi, y, 0.0, 24, trace=True); torch.cuda.synchronize()
        assert mp.mp_get_int("info_l2_bytes") == real // 4 and mp.mp_get_int("info_l2_pingpong") == 1
        want = 88.0 * (real / 132644864.0) / 4
        assert abs(mp.mp_get_int("info_l2_resident_mb") - want) <= 3, (mp.mp_get_int("info_l2_resident_mb"), want)
    finally:
        mp.mp_set_int("l2_bytes", 0); mp.mp_set_int("algo", 0)
    assert torch.equal(a.x, b.x) and torch.equal(a.r, b.r) and torch.equal(a.idx_trace, b.idx_trace) and torch.equal(a.c_trace, b.c_trace)


def test_two_host_threads_solve_at_once_with_the_same_bits(mp):
    """include/mp_b200.h: "with the knobs left alone, solves may be issued from several host threads".  Two threads, each with its
    own stream, outputs and workspace, solve their own cfg1-size signal 40 times while the other does the same (every launch
    reads the knobs and records its plan in the process-wide info_* fields, which are atomics); every result must be the bits
    of the same solve done alone."""
    import threading
    pb = problems.make_problem(problems.custom_config(256, 1024, 16, eps=1e-5, max_iter=128, B=2), seed=3)
    psi_d = dev(pb.psi32)
    ys = [dev(pb.Y[b]) for b in range(2)]
    alone = [mp.mp_recover(psi_d, ys[b], pb.cfg.eps, pb.cfg.max_iter, trace=True) for b in range(2)]
    torch.cuda.synchronize()
    assert all(int(a.n_iter.item()) > 0 for a in alone)
    errors = []

    def worker(b):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                ws = torch.empty(mp.mp_workspace_bytes(256, 1024, 1) + 256, dtype=torch.uint8, device="cuda")
                for _ in range(40):
                    got = mp.mp_recover(psi_d, ys[b], pb.cfg.eps, pb.cfg.max_iter, trace=True, workspace=ws, stream=s)
                    s.synchronize()
                    t = int(alone[b].n_iter.item())
                    ok = (int(got.n_iter.item()) == t and torch.equal(got.x, alone[b].x) and torch.equal(got.r, alone[b].r)
                          and torch.equal(got.idx_trace[:t], alone[b].idx_trace[:t]) and torch.equal(got.c_trace[:t], alone[b].c_trace[:t]))
                    if not ok:
                        errors.append(f"thread {b}: result differs from the solve done alone")
                        return
        except Exception as e:                                   # surfaced in the main thread below
            errors.append(f"thread {b}: {e!r}")

    threads = [threading.Thread(target=worker, args=(b,)) for b in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
    assert not any(t.is_alive() for t in threads), "a solver thread hangs"
    assert not errors, errors


def test_probe_read_reads_what_it_says_and_sums_what_it_read(mp):
    """mp_probe_read (the read-only ceiling bench.py quotes): the byte count it returns is k x 8 KiB x SMs x passes, a buffer below
    8 KiB per SM is refused, and the value left in `sink` is the weighted sum of exactly the floats it claims to have read (so the
    loads are real): with all-ones input each float4 contributes 1.0001 + 0.9999 + 1.0002 + 0.9998 = 4."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    unit = sms * 8192
    buf = torch.ones((3 * unit + 5000) // 4, dtype=torch.float32, device="cuda")
    sink = torch.zeros(1, dtype=torch.float32, device="cuda")
    read = mp.mp_probe_read(buf, 2, sink=sink)
    torch.cuda.synchronize()
    assert read == 3 * unit * 2
    assert abs(float(sink.item()) - read / 4.0) <= 2e-3 * read / 4.0          # fp32 accumulation of ~1.8 M ones per warp, summed by atomics
    with pytest.raises(mp.MPError) as e:
        mp.mp_probe_read(torch.ones(unit // 4 - 4, dtype=torch.float32, device="cuda"), 1, sink=sink)
    assert e.value.status == mp.MP_ERR_INVALID_ARG
    # and it is a bandwidth probe: a 64 MiB buffer read 50 times moves well above the HBM rate (it is served by L2)
    big = torch.ones((64 << 20) // 4, dtype=torch.float32, device="cuda")
    mp.mp_probe_read(big, 10, sink=sink); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); n = mp.mp_probe_read(big, 50, sink=sink); e1.record(); torch.cuda.synchronize()
    gbs = n / (e0.elapsed_time(e1) * 1e-3) / 1e9
    assert gbs > 9000, f"L2-resident probe reads only {gbs:.0f} GB/s"


def test_info_batched_algo_reports_the_path_taken(mp):
    """Auto dispatch may leave the tensor-core kernel (tiny dictionary, refused cooperative launch) and still return MP_OK:
    "info_batched_algo" is how a caller sees which kernel served the last batched call (1 lock-step, 2 sequential, 3 clusters)."""
    pb = problems.make_problem(problems.custom_config(128, 512, 6, max_iter=40, B=4), seed=9)
    psi_d, Y_d = dev(pb.psi32), dev(pb.Y)
    try:
        for knob, want in ((0, 3), (1, 1), (2, 2), (3, 3)):               # auto: 256 KiB dictionary -> one cluster per signal
            mp.mp_set_int("batched_algo", knob)
            res = mp.mp_recover_batched(psi_d, Y_d, pb.cfg.eps, pb.cfg.max_iter)
            torch.cuda.synchronize()
            assert mp.mp_get_int("info_batched_algo") == want, (knob, want)
            assert int(res.n_iter.min().item()) > 0
    finally:
        mp.mp_set_int("batched_algo", 0)
