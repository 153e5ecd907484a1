"""GPU parity of Orthogonal MP (mp_recover_omp) against the oracle's textbook OMP (normal equations,
Cholesky from scratch) fed the same fp32 bits.

Grading.  OMP's state is a function of the selected set alone (the coefficients are THE least-squares solution on it), so
the teacher-forced replay needs only the GPU's atom sequence: at every step the GPU's pick must be the oracle's argmax on
the oracle's own residual, or a near-tie (gap <= 1e-4 and |c_ref[pick]| >= (1 - 1e-4) max) -- the rule of the MP path.
Then x_gpu must be the least-squares solution on that set (1e-5 relative: QR in float64 on the GPU against normal
equations in float64 on the CPU, both rounded to fp32 once), r_gpu = y - Psi_S x_S to 1e-6 ||r|| + 1e-11 ||y|| (fp32 rounding of the output, float64 refit on both sides), the stop
rule must hold on the replay's norms, and when no near-tie occurred the free-running oracle takes the same atoms."""
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
    m.mp_set_int("chunk", 64)
    m.mp_set_int("omp_algo", 0)


OMP_ALGOS = [1, 2]        # 1 = one persistent kernel (basis slices stationary in shared memory), 2 = stream loop of small kernels


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run(mp, psi32, y32, eps, max_iter, ld=None, algo=0):
    mp.mp_set_int("omp_algo", algo)
    M, N = psi32.shape
    if ld is None:
        ld = (N + 3) // 4 * 4
    buf = torch.full((M, ld), 7.0, dtype=torch.float32, device="cuda"); buf[:, :N] = dev(psi32)
    res = mp.mp_recover_omp(buf[:, :N], dev(y32), eps, max_iter, trace=True)
    torch.cuda.synchronize()
    t = int(res.n_iter.item())
    return res.x.cpu().numpy().astype(np.float64), res.r.cpu().numpy().astype(np.float64), t, res.idx_trace.cpu().numpy()[:t]


def grade_omp(psi32, y32, eps, max_iter, x, r, t, idx, x_true=None, support=None):
    th = oracle.default_threads()
    eps = float(np.float32(eps))
    y = y32.astype(np.float64)
    M, N = psi32.shape
    assert 0 <= t <= min(max_iter, N) and len(set(idx.tolist())) == t, "an atom was taken twice"
    rp = oracle.omp(psi32, y, 0.0, 0, idx_force=idx, nthreads=th)
    assert rp.status == 0 and rp.n_iter == t
    same = idx == rp.argmax_ref
    legal = same | ((rp.gap <= grading.GAP_TOL) & (np.abs(rp.c_at_idx) >= (1 - grading.GAP_TOL) * rp.cmax_ref))
    assert legal.all(), f"illegal pick at t={int(np.nonzero(~legal)[0][0])}"
    nx = np.linalg.norm(rp.x)
    assert np.linalg.norm(x - rp.x) <= 1e-5 * nx + 1e-30, f"x is not the least-squares solution: {np.linalg.norm(x - rp.x) / max(nx, 1e-300):.2e}"
    off = np.ones(M, bool); off[idx] = False
    assert not x[off].any()
    nr = rp.rnorm[t]
    assert np.linalg.norm(r - rp.r) <= 1e-6 * nr + 1e-11 * np.linalg.norm(y) + 1e-30, "r is not y - Psi_S x_S"
    thr = eps * rp.rnorm[0]
    if t:
        assert np.all(rp.rnorm[:t] > thr * (1 - 1e-6)), "GPU continued although ||r|| <= eps ||y||"
    if t < min(max_iter, N):
        assert rp.rnorm[t] <= thr * (1 + 1e-6), "GPU stopped although ||r|| > eps ||y|| and t < T"
    ref = oracle.omp(psi32, y, eps, max_iter, nthreads=th)
    if same.all() and not np.any(ref.gap <= grading.GAP_TOL):
        assert t == ref.n_iter and np.array_equal(idx, ref.idx)
    if x_true is not None and support is not None and np.linalg.norm(ref.x - x_true) <= 1e-4 * np.linalg.norm(x_true):
        assert set(idx.tolist()) <= set(int(s) for s in support)
        assert np.linalg.norm(x - x_true) <= 1e-4 * np.linalg.norm(x_true)
    return ref


@pytest.mark.parametrize("algo", OMP_ALGOS)
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_cfg1_omp_full_grading(mp, seed, algo):
    pb = problems.make_problem(synth.config("cfg1"), seed)
    c = pb.cfg
    x, r, t, idx = run(mp, pb.psi32, pb.Y[0], c.eps, c.max_iter, algo=algo)
    assert mp.mp_get_int("info_omp_algo") == algo
    ref = grade_omp(pb.psi32, pb.Y[0], c.eps, c.max_iter, x, r, t, idx, x_true=pb.X[0], support=pb.S[0])
    assert t <= c.K and ref.n_iter == t                                      # OMP: one step per atom of the support


@pytest.mark.parametrize("N,M,K,ld", [(250, 1000, 10, None), (37, 5, 2, 40), (1, 3, 1, 4), (130, 149, 6, 256),
                                      (2052, 777, 20, None), (512, 4099, 24, None)])
@pytest.mark.parametrize("algo", OMP_ALGOS)
def test_ragged_shapes_omp(mp, N, M, K, ld, algo):
    cfg = problems.custom_config(N, M, K, eps=1e-4, max_iter=3 * K + 3)
    pb = problems.make_problem(cfg, seed=4)
    x, r, t, idx = run(mp, pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, ld, algo=algo)
    grade_omp(pb.psi32, pb.Y[0], cfg.eps, cfg.max_iter, x, r, t, idx)


@pytest.mark.parametrize("algo", OMP_ALGOS)
def test_edge_cases_omp(mp, algo):
    pb = problems.make_problem(problems.custom_config(64, 200, 4), seed=2)
    y = pb.Y[0]
    x, r, t, _ = run(mp, pb.psi32, np.zeros_like(y), 1e-5, 50, algo=algo)
    assert t == 0 and not x.any() and not r.any()
    x, r, t, _ = run(mp, pb.psi32, y, 1e-5, 0, algo=0)
    assert t == 0 and not x.any() and np.array_equal(r.astype(np.float32), y)
    x, r, t, _ = run(mp, pb.psi32, y, 1.0, 50, algo=algo)
    assert t == 0
    mp.mp_set_int("chunk", 3)                                                # several host polls
    pb2 = problems.make_problem(problems.custom_config(64, 200, 30), seed=3)
    x, r, t, idx = run(mp, pb2.psi32, pb2.Y[0], 0.0, 20, algo=algo)          # eps = 0: runs to max_iter
    mp.mp_set_int("chunk", 64)
    assert t == 20
    grade_omp(pb2.psi32, pb2.Y[0], 0.0, 20, x, r, t, idx)
    x, r, t, idx = run(mp, pb2.psi32, pb2.Y[0], 0.0, 1000, algo=algo)        # capped at N atoms
    assert t <= 64


@pytest.mark.parametrize("algo", OMP_ALGOS)
def test_omp_equals_mp_on_orthonormal_dictionary(mp, algo):
    N = 256
    H = np.array([[1.0]])
    while H.shape[0] < N:
        H = np.block([[H, H], [H, -H]])
    psi = (H / 16.0).astype(np.float32)
    rng = np.random.default_rng(5)
    s = rng.choice(N, 12, replace=False)
    x_true = np.zeros(N); x_true[s] = rng.standard_normal(12)
    y = (psi.astype(np.float64).T @ x_true).astype(np.float32)
    x, r, t, idx = run(mp, psi, y, 1e-6, 100, algo=algo)
    assert t == 12 and list(idx) == list(s[np.argsort(-np.abs(x_true[s]), kind="stable")])
    assert np.allclose(x, x_true, atol=2e-7)


@pytest.mark.parametrize("algo", OMP_ALGOS)
def test_cfg2_size_omp(mp, algo):
    """N=2048, M=8192, K=128: OMP takes exactly the support in K steps; the replay grades every step."""
    pb = problems.make_problem(synth.config("cfg2"), 1)
    c = pb.cfg
    x, r, t, idx = run(mp, pb.psi32, pb.Y[0], c.eps, 4 * c.K, algo=algo)
    assert t == c.K and set(idx.tolist()) == set(pb.S[0].tolist())
    grade_omp(pb.psi32, pb.Y[0], c.eps, 4 * c.K, x, r, t, idx, x_true=pb.X[0], support=pb.S[0])


@pytest.mark.parametrize("a", [2.0, 5.0])
@pytest.mark.parametrize("algo", OMP_ALGOS)
def test_coherent_dictionary_omp(mp, a, algo):
    """Atoms share a strong common component (pairwise coherence a^2/(a^2+1) = 0.8 / 0.96): after the first pick the
    Gram-Schmidt step removes more than half of every later atom, which is where a single pass loses orthogonality and the
    persistent kernel's second pass has to run.  Same grading as everywhere: picks against the oracle's normal-equation OMP,
    x = the least-squares solution on the selected set, r = y - Psi_S x_S."""
    N, M, K = 300, 640, 8
    rng = np.random.default_rng(11)
    u = rng.standard_normal(N); u /= np.linalg.norm(u)
    raw = (a * u[None, :] + rng.standard_normal((M, N)) / np.sqrt(N)).astype(np.float32)
    psi32 = problems.normalise_on_host(raw)
    s = rng.choice(M, K, replace=False)
    x_true = np.zeros(M); x_true[s] = rng.standard_normal(K)
    y = (psi32.astype(np.float64).T @ x_true).astype(np.float32)
    x, r, t, idx = run(mp, psi32, y, 1e-5, 4 * K, algo=algo)
    assert t >= 2
    grade_omp(psi32, y, 1e-5, 4 * K, x, r, t, idx)
