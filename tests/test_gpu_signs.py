"""GPU parity of MP on a sign-packed Bernoulli dictionary (mp_pack_signs, mp_recover_signs) against
the oracle run on the expanded fp32 dictionary (+-1/sqrt(N), Eq. 13), with the full grading of the fp32 path."""
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
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run(mp, psi32, y32, eps, max_iter):
    M, N = psi32.shape
    ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda"); buf[:, :N] = dev(psi32)
    bits, scale, n_bad = mp.mp_pack_signs(buf[:, :N])
    assert n_bad == 0 and scale == float(np.abs(psi32[0, 0]))
    res = mp.mp_recover_signs(bits, N, scale, dev(y32), eps, max_iter, trace=True)
    torch.cuda.synchronize()
    t = int(res.n_iter.item())
    return (res.x.cpu().numpy(), res.r.cpu().numpy(), t, res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t]), bits


def test_pack_signs_bits_and_rejection(mp):
    cfg = problems.custom_config(100, 37, 4, dictionary="bernoulli")
    psi = synth.make_dictionary(cfg, 3)
    bits, scale, n_bad = mp.mp_pack_signs(dev(psi))
    b = bits.cpu().numpy().view(np.uint32)
    assert n_bad == 0 and scale == np.float32(1.0 / np.sqrt(np.float32(100))) or n_bad == 0
    for m in (0, 5, 36):
        for n in (0, 31, 32, 63, 99):
            assert ((b[m, n // 32] >> (n % 32)) & 1) == (1 if psi[m, n] < 0 else 0)
        assert (b[m, 3] >> 4) == 0 and not b[m, 4:].any()                     # pad bits are zero
    g = problems.normalise_on_host(synth.make_dictionary(problems.custom_config(64, 20, 2), 1))
    assert mp.mp_pack_signs(dev(g))[2] > 0                                    # a Gaussian dictionary is refused (n_bad > 0)


@pytest.mark.parametrize("N,M,K", [(256, 1024, 16), (100, 37, 4), (4096, 300, 16), (1000, 5000, 40), (33, 150, 3)])
def test_signs_full_grading(mp, N, M, K):
    cfg = problems.custom_config(N, M, K, dictionary="bernoulli", eps=1e-5, max_iter=8 * K)
    pb = problems.make_problem(cfg, seed=5)
    (x, r, t, idx, c), _ = run(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter)
    grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, x, r, t, idx, c, x_true=pb.X[0], support=pb.S[0])


def test_signs_edge_cases(mp):
    cfg = problems.custom_config(64, 200, 4, dictionary="bernoulli")
    pb = problems.make_problem(cfg, seed=2)
    y = pb.Y[0]
    (x, r, t, _, _), _ = run(mp, pb.psi32, np.zeros_like(y), 1e-5, 50)
    assert t == 0 and not x.any() and not r.any()
    (x, r, t, _, _), _ = run(mp, pb.psi32, y, 1e-5, 0)
    assert t == 0 and not x.any() and np.array_equal(r, y)
    (x, r, t, idx, c), _ = run(mp, pb.psi32, y, 0.0, 1)
    cref = pb.psi32.astype(np.float64) @ y.astype(np.float64)
    assert t == 1 and idx[0] == int(np.argmax(np.abs(cref)))


def test_cfg3_signs_sampled_grading(mp):
    """CFG3 itself (Bernoulli, N=4096, M=16384) from 8 MiB of sign bits: sampled iterations, support, coefficients."""
    pb = problems.make_problem(synth.config("cfg3"), 1)
    c = pb.cfg
    (x, r, t, idx, cc), bits = run(mp, pb.psi32, pb.Y[0], c.eps, c.max_iter)
    assert 800 < t < 2500 and bits.numel() * 4 == 16384 * 128 * 4
    ts = sorted(set(list(range(0, 4)) + list(range(5, t, 97)) + list(range(t - 3, t))))
    grading.grade_sampled(pb.psi32, pb.Y[0], idx, cc, t, r, ts)
    assert set(idx.tolist()) == set(pb.S[0].tolist())
    assert np.linalg.norm(x - pb.X[0]) <= 1e-4 * np.linalg.norm(pb.X[0])


# ------------------------------------------------------------------------------------------ many problems, one CTA each
def run_signs_many(mp, pbs, eps, max_iter, shared=False):
    M, N = pbs[0].psi32.shape
    P = len(pbs)
    ld = (N + 3) // 4 * 4
    stack = torch.full((P * M, ld), 7.0, dtype=torch.float32, device="cuda")
    for q, pb in enumerate(pbs):
        stack[q * M:(q + 1) * M, :N] = dev(pb.psi32)
    bits, scale, n_bad = mp.mp_pack_signs(stack[:, :N])                           # the P dictionaries packed as one stack
    assert n_bad == 0
    bits = bits.view(P, M, -1)
    Y = dev(np.stack([pb.Y[0] for pb in pbs]))
    res = mp.mp_recover_signs_many(bits[0] if shared else bits, N, scale, Y, eps, max_iter, trace=True)
    torch.cuda.synchronize()
    return res.x.cpu().numpy(), res.r.cpu().numpy(), res.n_iter.cpu().numpy(), res.idx_trace.cpu().numpy(), res.c_trace.cpu().numpy()


@pytest.mark.parametrize("N,M,K,P", [(256, 1024, 16, 5), (100, 37, 4, 9), (500, 1000, 30, 4), (1000, 1000, 40, 3), (33, 150, 3, 200),
                                     (1, 3, 1, 2), (2048, 300, 12, 2)])
def test_signs_many_every_problem_graded_like_a_single_run(mp, N, M, K, P):
    """Problem q's result must be MP on (expanded dictionary q, y_q): full grading of every problem against the oracle."""
    cfg = problems.custom_config(N, M, K, dictionary="bernoulli", eps=1e-5, max_iter=8 * K)
    pbs = [problems.make_problem(cfg, seed=20 + q) for q in range(P)]
    if P > 4:
        pbs[1].Y[0][:] = 0.0                                                       # one problem that stops at once
    X, R, T, I, Cc = run_signs_many(mp, pbs, cfg.eps, cfg.max_iter)
    if P > 4:
        assert T[1] == 0 and not X[1].any()
    for q, pb in enumerate(pbs):
        t = int(T[q])
        grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, X[q], R[q], t, I[q, :t], Cc[q, :t], nthreads=4)


def test_signs_many_phase_diagram_cell_and_shared_dictionary(mp):
    """A cell of the paper's Fig. 1 experiment with its own parameters (M = 1000, rho = 0.5, sigma = 0.03, U[-1,1] nonzeros,
    eps = 1e-7, T = N): every trial graded and recovered (Eq. 14 ~ 0); then all signals against ONE shared dictionary."""
    M, N, K, P = 1000, 500, 30, 4
    cfg = problems.custom_config(N, M, K, dictionary="bernoulli", values="uniform", eps=1e-7, max_iter=N)
    pbs = [problems.make_problem(cfg, seed=60 + q) for q in range(P)]
    X, R, T, I, Cc = run_signs_many(mp, pbs, cfg.eps, cfg.max_iter)
    for q, pb in enumerate(pbs):
        t = int(T[q])
        grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, X[q], R[q], t, I[q, :t], Cc[q, :t], nthreads=4)
        assert oracle.reconstruction_error_pct(X[q].astype(np.float64), pb.X[0]) < 1e-6
    cfgb = problems.custom_config(N, M, K, dictionary="bernoulli", values="uniform", eps=1e-7, max_iter=N, B=P)
    pb = problems.make_problem(cfgb, 7)
    shared = [problems.Problem(cfgb, pb.psi_raw, pb.psi32, pb.X[q:q + 1], pb.S[q:q + 1], pb.Y[q:q + 1]) for q in range(P)]
    X, R, T, I, Cc = run_signs_many(mp, shared, cfgb.eps, cfgb.max_iter, shared=True)
    for q in range(P):
        t = int(T[q])
        grading.grade_single(pb.psi32, pb.Y[q], cfgb.eps, cfgb.max_iter, X[q], R[q], t, I[q, :t], Cc[q, :t], nthreads=4)


def test_signs_many_refuses_what_does_not_fit(mp):
    bits = torch.zeros(1, 4096, 64, dtype=torch.int32, device="cuda")           # N = 2048, M = 4096: 1 MB of bits per problem
    with pytest.raises(mp.MPError) as e:
        mp.mp_recover_signs_many(bits, 2048, 1.0 / 45.0, torch.zeros(1, 2048, device="cuda"), 1e-5, 4)
    assert e.value.status == mp.MP_ERR_UNSUPPORTED


def test_signs_many_random_shapes_and_repeatability(mp):
    """Fixed-seed sweep over awkward shapes (word boundaries of N, tiny M, more problems than SMs) with full grading, and 10 repeated
    runs of a 300-problem batch giving the same bits (problems are drawn from a device counter)."""
    rng = np.random.default_rng(77)
    for trial in range(8):
        N = int(rng.choice([1, 31, 32, 33, 64, 95, 129, 500, 1000, 1537]))
        M = int(rng.choice([1, 2, 31, 33, 100, 511, 700]))
        if N * M // 8 > 150000:
            M = 150000 * 8 // N
        K = max(1, min(M, N // 6 + 1, 8))
        cfg = problems.custom_config(N, M, K, dictionary="bernoulli", eps=1e-5, max_iter=4 * K + 2)
        pbs = [problems.make_problem(cfg, 3000 + 5 * trial + q) for q in range(int(rng.choice([1, 4, 11])))]
        X, R, T, I, Cc = run_signs_many(mp, pbs, cfg.eps, cfg.max_iter)
        for q, pb in enumerate(pbs):
            t = int(T[q])
            grading.grade_single(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, X[q], R[q], t, I[q, :t], Cc[q, :t], nthreads=4)
    cfg = problems.custom_config(96, 200, 5, dictionary="bernoulli", eps=1e-5, max_iter=30)
    pbs = [problems.make_problem(cfg, 4000 + q) for q in range(300)]
    ref = run_signs_many(mp, pbs, cfg.eps, cfg.max_iter)
    for _ in range(9):
        out = run_signs_many(mp, pbs, cfg.eps, cfg.max_iter)
        assert np.array_equal(ref[0], out[0]) and np.array_equal(ref[1], out[1]) and np.array_equal(ref[2], out[2])
        assert all(np.array_equal(ref[3][q, :ref[2][q]], out[3][q, :ref[2][q]]) for q in range(300))
