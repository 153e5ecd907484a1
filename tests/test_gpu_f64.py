"""GPU parity of the double-precision path (mp_recover_f64, mp_normalize_columns_f64) against the
float64 oracle fed the same float64 bits.  All arithmetic is float64 on both sides, so the tolerances are those of
reordered float64 sums, not the fp32 ones of tests/grading.py: step values to 1e-10 ||r|| (||r|| falls to 1e-5 ||y||, and the float64 state itself is only known to ~1e-16 ||y||), the residual vector to
1e-10 relative, coefficients to 1e-14."""
import numpy as np
import pytest
import torch

import oracle
from paper_0809_1833_b200 import synth
import grading
import problems

pytestmark = pytest.mark.gpu
EPS = float(np.float32(1e-5))            # exactly the value both sides use


@pytest.fixture(scope="module")
def mp():
    import paper_0809_1833_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_f64(N, M, K, seed, dictionary="gaussian"):
    cfg = problems.custom_config(N, M, K, dictionary=dictionary)
    raw = synth.make_dictionary(cfg, seed).astype(np.float64)
    psi, _ = oracle.normalize_columns(raw)                                   # float64, not rounded
    x, s = synth.sparse_signal(M, K, seed, "normal", signal=0)
    y = np.zeros(N)
    for m in np.sort(s):
        y += x[m] * psi[m]
    return psi, x, s, y


def run(mp, psi, y, eps, max_iter, ld=None):
    M, N = psi.shape
    if ld is None:
        ld = (N + 1) // 2 * 2
    buf = torch.full((M, ld), 7.0, dtype=torch.float64, device="cuda")       # pad columns hold garbage on purpose
    buf[:, :N] = dev(psi)
    res = mp.mp_recover_f64(buf[:, :N], dev(y), eps, max_iter, trace=True)
    torch.cuda.synchronize()
    t = int(res.n_iter.item())
    return res.x.cpu().numpy(), res.r.cpu().numpy(), t, res.idx_trace.cpu().numpy()[:t], res.c_trace.cpu().numpy()[:t]


def grade(psi, y, eps, max_iter, x, r, t, idx, c, **kw):
    g = grading.grade_single(psi, y, eps, max_iter, x, r, t, idx, c, c_tol=1e-10, **kw)
    rp = oracle.mp_replay(psi, y, idx, c, oracle.default_threads())
    assert np.linalg.norm(r - rp.r) <= 1e-10 * np.linalg.norm(rp.r) + 1e-300
    assert np.all(np.abs(x - rp.x) <= 1e-14 * np.abs(rp.x) + 1e-300)
    return g


@pytest.mark.parametrize("N,M", [(256, 1024), (251, 33), (1, 5), (4096, 300)])
def test_normalize_columns_f64(mp, N, M):
    rng = np.random.default_rng(1)
    raw = rng.standard_normal((M, N))
    raw[M // 2] = 0.0                                                        # a zero atom stays zero (R7)
    ld = N + 3
    buf = torch.full((M, ld), 5.0, dtype=torch.float64, device="cuda"); buf[:, :N] = dev(raw)
    norms = torch.empty(M, dtype=torch.float64, device="cuda")
    mp.mp_normalize_columns_f64(buf[:, :N], norms)
    torch.cuda.synchronize()
    ref, nref = oracle.normalize_columns(raw)
    got = buf[:, :N].cpu().numpy()
    assert np.allclose(norms.cpu().numpy(), nref, rtol=1e-14, atol=0)
    assert np.allclose(got, ref, rtol=1e-14, atol=1e-300) and not got[M // 2].any()
    assert torch.all(buf[:, N:] == 5.0)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_cfg1_shape_full_grading_f64(mp, seed):
    psi, x_true, s, y = make_f64(256, 1024, 16, seed)
    x, r, t, idx, c = run(mp, psi, y, EPS, 4096)
    g = grade(psi, y, EPS, 4096, x, r, t, idx, c, x_true=x_true, support=s)
    assert g.exact_recovery and g.first_divergence == -1 and g.n_iter_gpu == g.n_iter_ref


@pytest.mark.parametrize("N,M,K,ld", [(251, 1000, 10, None), (37, 5, 2, 40), (1, 3, 1, 2), (131, 149, 6, 256),
                                      (2053, 777, 20, None), (8192, 320, 16, None), (512, 4099, 24, None)])
def test_ragged_shapes_f64(mp, N, M, K, ld):
    psi, x_true, s, y = make_f64(N, M, K, 4)
    T = 6 * K + 3
    x, r, t, idx, c = run(mp, psi, y, 1e-4, T, ld)
    grade(psi, y, 1e-4, T, x, r, t, idx, c)


def test_edge_cases_f64(mp):
    psi, _, _, y = make_f64(64, 200, 4, 2)
    x, r, t, _, _ = run(mp, psi, np.zeros_like(y), EPS, 50)
    assert t == 0 and not x.any() and not r.any()
    x, r, t, _, _ = run(mp, psi, y, EPS, 0)
    assert t == 0 and not x.any() and np.array_equal(r, y)
    x, r, t, _, _ = run(mp, psi, y, 1.0, 50)
    assert t == 0 and np.array_equal(r, y)
    psi2, _, _, y2 = make_f64(64, 200, 24, 3)                               # K too large to converge: stays above the rounding floor
    x, r, t, idx, c = run(mp, psi2, y2, 0.0, 40)
    assert t == 40 and np.linalg.norm(r) > 1e-6 * np.linalg.norm(y2)
    grade(psi2, y2, 0.0, 40, x, r, t, idx, c)
    x, r, t, idx, c = run(mp, psi, y, 0.0, 1)
    cref = psi @ y
    assert t == 1 and idx[0] == int(np.argmax(np.abs(cref))) and abs(c[0] - cref[idx[0]]) <= 1e-14 * np.linalg.norm(y)


def test_orthonormal_hadamard_f64(mp):
    """Orthonormal Psi (Sylvester-Hadamard / sqrt(N), N a power of 4: entries exact): K-sparse x recovered in exactly K
    steps in order of decreasing |x|, residual exactly representable steps."""
    N = 256
    H = np.array([[1.0]])
    while H.shape[0] < N:
        H = np.block([[H, H], [H, -H]])
    psi = H / 16.0
    rng = np.random.default_rng(5)
    s = rng.choice(N, 12, replace=False)
    x_true = np.zeros(N); x_true[s] = rng.standard_normal(12)
    y = psi.T @ x_true
    x, r, t, idx, c = run(mp, psi, y, 1e-12, 100)
    assert t == 12 and list(idx) == list(s[np.argsort(-np.abs(x_true[s]), kind="stable")])
    assert np.allclose(x, x_true, atol=1e-14) and np.linalg.norm(r) <= 1e-14 * np.linalg.norm(y)


def test_tie_break_lowest_index_f64(mp):
    rng = np.random.default_rng(7)
    psi = rng.standard_normal((300, 64)); psi /= np.linalg.norm(psi, axis=1, keepdims=True)
    psi[200] = psi[17]; psi[250] = -psi[17]                                  # duplicated and negated atoms: always min index
    y = 3.0 * psi[17]
    x, r, t, idx, c = run(mp, psi, y, 1e-12, 5)
    assert idx[0] == 17 and abs(c[0] - 3.0) < 1e-14


def test_cfg2_size_sampled_grading_f64(mp):
    """N=2048, M=8192 in double (128 MiB): sampled iterations rebuilt in float64 from the trace, final residual, support."""
    psi, x_true, s, y = make_f64(2048, 8192, 128, 1)
    x, r, t, idx, c = run(mp, psi, y, EPS, 16384)
    assert 400 < t < 1500
    ts = sorted(set(list(range(0, 3)) + list(range(5, t, 61)) + list(range(t - 3, t))))
    out = grading.grade_sampled(psi, y, idx, c, t, r, ts, c_tol=1e-10)
    assert set(idx.tolist()) <= set(s.tolist())
    assert np.linalg.norm(x - x_true) <= 1e-4 * np.linalg.norm(x_true)
    assert np.linalg.norm(r) <= EPS * np.linalg.norm(y) * (1 + 1e-9)
