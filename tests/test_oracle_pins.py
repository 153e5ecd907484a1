"""Pins for the CPU oracle (oracle/mp_oracle.c) against what the paper and the mathematics
fix -- NOT against itself.  Each test names the passage of PAPER.md ("P:n") or the closed
form it checks.  A plausible mistake anywhere in the oracle (dropped term, wrong sign or
index, transposed operand, wrong tie-break, stale norm) fails at least one of these.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_0809_1833_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- helpers
def hadamard(n):
    H = np.array([[1.0]])
    while H.shape[0] < n:
        H = np.block([[H, H], [H, -H]])
    assert H.shape[0] == n
    return H


def orthonormal_cases():
    rng = np.random.default_rng(7)
    out = {}
    out["identity"] = np.eye(12)
    P = np.eye(12)[rng.permutation(12)] * rng.choice([-1.0, 1.0], 12)[None, :]
    out["signed_permutation"] = P
    out["hadamard16"] = hadamard(16) / 4.0            # entries +-1/4 exactly representable
    out["hadamard64"] = hadamard(64) / 8.0
    v = rng.standard_normal(20)
    v /= np.linalg.norm(v)
    out["householder"] = np.eye(20) - 2.0 * np.outer(v, v)
    Q, _ = np.linalg.qr(rng.standard_normal((24, 24)))
    out["qr_gaussian"] = Q
    return out


def psi_t_of(Psi):
    """paper's N x M matrix -> atom-major [M, N] C-contiguous"""
    return np.ascontiguousarray(Psi.T)


# ----------------------------------------------------------------------------- whole loop, exact case
@pytest.mark.parametrize("name", list(orthonormal_cases().keys()))
def test_orthonormal_dictionary_recovers_k_sparse_in_k_steps(name):
    """BASELINE north_star / Eq. 8-12: with Psi orthonormal (N=M), c = x on the first pass, atoms
    are taken in order of decreasing |x_m|, n_iter = K exactly, x~ = x, r = 0."""
    Psi = orthonormal_cases()[name]
    n = Psi.shape[0]
    rng = np.random.default_rng(3)
    K = 5
    S = rng.choice(n, K, replace=False)
    x = np.zeros(n)
    x[S] = rng.standard_normal(K) + np.sign(rng.standard_normal(K)) * 0.5   # distinct magnitudes, none tiny
    y = Psi @ x
    res = oracle.mp(psi_t_of(Psi), y, 1e-12, 100)
    assert res.n_iter == K
    order = S[np.argsort(-np.abs(x[S]), kind="stable")]
    assert list(res.idx) == list(order)
    np.testing.assert_allclose(res.x, x, atol=1e-14, rtol=0)
    assert np.linalg.norm(res.r) <= 1e-14 * np.linalg.norm(y)
    np.testing.assert_allclose(res.c, x[order], atol=1e-14, rtol=0)


def test_identity_dictionary_exact_zero_residual_with_eps_zero():
    """Identity/permutation: r becomes EXACTLY 0 after K steps so even eps = 0 stops (0 > 0 false)."""
    x = np.zeros(10)
    x[[2, 7, 4]] = [1.5, -3.0, 0.25]
    res = oracle.mp(psi_t_of(np.eye(10)), x.copy(), 0.0, 50)
    assert res.n_iter == 3 and list(res.idx) == [7, 2, 4]
    assert np.all(res.r == 0.0) and np.array_equal(res.x, x)


# ----------------------------------------------------------------------------- non-orthogonal dynamics, closed form
@pytest.mark.parametrize("mu", [0.5, -0.5, 0.9])
def test_two_atoms_residual_contracts_by_coherence(mu):
    """Two unit atoms with <psi0,psi1> = mu and y in their span: after the first step MP alternates
    atoms and ||r_{t+1}|| = |mu| ||r_t|| exactly (r_t is orthogonal to the atom just used, so
    <r_t,psi_j>^2 = ||r_t||^2 (1-mu^2)).  Follows from Eq. 9-11 alone."""
    N = 5
    psi0 = np.zeros(N); psi0[0] = 1.0
    psi1 = np.zeros(N); psi1[0] = mu; psi1[1] = math.sqrt(1 - mu * mu)
    a, b = 2.0, 0.7
    y = a * psi0 + b * psi1
    eps = 1e-9
    res = oracle.mp(np.stack([psi0, psi1]), y, eps, 10_000)
    rn = res.rnorm
    assert res.idx[0] == 0                      # |<y,psi0>| = |a + b mu| > |<y,psi1>| = |a mu + b|
    assert all(res.idx[t] != res.idx[t + 1] for t in range(res.n_iter - 1))
    ratios = rn[2:] / rn[1:-1]
    np.testing.assert_allclose(ratios[: 40], abs(mu), rtol=1e-9)
    # n_iter = 1 + ceil( log(eps||y||/||r_1||) / log|mu| )
    expect = 1 + math.ceil(math.log(eps * rn[0] / rn[1]) / math.log(abs(mu)))
    assert abs(res.n_iter - expect) <= 1
    np.testing.assert_allclose(res.x, [a, b], atol=1e-7)


def test_single_atom_is_orthogonal_projection():
    """M = 1: x~_0 = <y,psi_0>, r = y - x~_0 psi_0, and the second pass finds c ~ 0."""
    rng = np.random.default_rng(0)
    psi = rng.standard_normal(9); psi /= np.linalg.norm(psi)
    y = rng.standard_normal(9)
    res = oracle.mp(psi[None, :], y, 0.0, 2)
    assert res.n_iter == 2
    assert res.c[0] == pytest.approx(float(y @ psi), rel=1e-15)
    assert abs(res.c[1]) <= 1e-15 * np.linalg.norm(y)
    np.testing.assert_allclose(res.r, y - (y @ psi) * psi, atol=1e-15)


def test_one_iteration_equals_textbook_gemv_and_argmax():
    """max_iter = 1 on any input = one matrix-vector product + arg-abs-max (Eq. 15-16);
    numpy's float64 routines are the independent textbook implementation.  N != M so a transposed
    operand cannot pass."""
    rng = np.random.default_rng(11)
    N, M = 37, 91
    Psi = rng.standard_normal((N, M))
    Psi /= np.linalg.norm(Psi, axis=0, keepdims=True)
    y = rng.standard_normal(N)
    res = oracle.mp(psi_t_of(Psi), y, 0.0, 1)
    c = Psi.T @ y
    i = int(np.argmax(np.abs(c)))
    assert res.n_iter == 1 and res.idx[0] == i
    assert res.c[0] == pytest.approx(c[i], rel=1e-13)
    np.testing.assert_allclose(res.r, y - c[i] * Psi[:, i], atol=1e-13)
    x = np.zeros(M); x[i] = c[i]
    np.testing.assert_allclose(res.x, x, atol=1e-13)
    np.testing.assert_allclose(oracle.correlate(psi_t_of(Psi), y), c, atol=1e-13)


# ----------------------------------------------------------------------------- argmax and tie-break
def test_argmax_matches_brute_force_on_tiny_inputs():
    """north_star: on tiny inputs (M <= 16) each argmax must match a brute-force scan."""
    rng = np.random.default_rng(5)
    for trial in range(200):
        M = int(rng.integers(1, 17))
        c = rng.standard_normal(M)
        if trial % 3 == 0:                        # inject exact ties, signs mixed
            j, k = rng.integers(0, M, 2)
            c[k] = -c[j]
        best = max(abs(v) for v in c)
        brute = min(m for m in range(M) if abs(c[m]) == best)
        assert oracle.argmax_abs(c) == brute


def test_argmax_tie_breaks_to_lowest_index_and_nan_never_wins():
    """P:144 'the smallest index of the maximum magnitude element'."""
    assert oracle.argmax_abs([1.0, -2.0, 2.0, -2.0]) == 1
    assert oracle.argmax_abs([0.0, -0.0, 0.0]) == 0
    assert oracle.argmax_abs([float("nan"), 1.0, 3.0]) == 2
    assert oracle.argmax_abs([3.0, float("nan"), 3.0]) == 0


def test_duplicate_and_negated_atoms_pick_the_lower_index():
    rng = np.random.default_rng(2)
    N, M = 16, 12
    Psi = rng.standard_normal((N, M)); Psi /= np.linalg.norm(Psi, axis=0)
    y = Psi[:, 8] * 3.0 + 0.01 * rng.standard_normal(N)
    for sign in (+1.0, -1.0):
        P2 = Psi.copy()
        P2[:, 3] = sign * P2[:, 8]                 # atom 3 == +-atom 8
        res = oracle.mp(psi_t_of(P2), y, 0.0, 1)
        assert res.idx[0] == 3
        assert res.c[0] == pytest.approx(sign * float(y @ Psi[:, 8]), rel=1e-14)


def test_all_equal_correlations_pick_index_zero():
    """Psi = Hadamard/sqrt(N), y = e_0: every c_m = 1/sqrt(N) exactly."""
    H = hadamard(16) / 4.0
    y = np.zeros(16); y[0] = 1.0
    res = oracle.mp(psi_t_of(H), y, 0.0, 1)
    assert res.idx[0] == 0 and res.c[0] == 0.25 and res.gap[0] == 0.0


# ----------------------------------------------------------------------------- every iteration, any input
def _random_problem(seed, N=48, M=160, K=6, dtype=np.float64):
    raw = synth.gaussian_dictionary(N, M, seed).astype(np.float64)
    psi_t, _ = oracle.normalize_columns(raw)
    x, S = synth.sparse_signal(M, K, seed, "normal")
    y = (psi_t.T @ x)
    return psi_t.astype(dtype), x, S, y


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_per_iteration_invariants(seed):
    psi_t, x_true, S, y = _random_problem(seed)
    res = oracle.mp(psi_t, y, 1e-9, 400)
    assert 0 < res.n_iter < 400
    rn, c, idx = res.rnorm, res.c, res.idx
    col_sq = np.sum(psi_t * psi_t, axis=1)
    # (1) energy identity ||r'||^2 = ||r||^2 - c^2 (2 - ||psi_i||^2)  [= ||r||^2 - c^2 for unit columns, north_star]
    lhs = rn[1:] ** 2
    rhs = rn[:-1] ** 2 - c * c * (2.0 - col_sq[idx])
    assert np.all(np.abs(lhs - rhs) <= 1e-12 * rn[:-1] ** 2)
    # (2) ||r|| non-increasing (north_star)
    assert np.all(np.diff(rn) <= 0.0)
    # (5) Cauchy-Schwarz |c_i| <= ||r|| ||psi_i||
    assert np.all(np.abs(c) <= rn[:-1] * np.sqrt(col_sq[idx]) * (1 + 1e-12))
    # (4) consistency: r == y - Psi x~ recomputed from scratch
    assert np.linalg.norm((y - psi_t.T @ res.x) - res.r) <= 1e-13 * np.linalg.norm(y)
    # x~ is the sum of the steps per atom (Eq. 10)
    x_from_trace = np.zeros_like(res.x)
    np.add.at(x_from_trace, idx, c)
    np.testing.assert_allclose(res.x, x_from_trace, atol=1e-14)
    # stop rule: last recorded norm is at/below threshold, the one before is above
    assert rn[-1] <= 1e-9 * rn[0] < rn[-2]
    # exact-recovery regime: x~ -> x
    assert np.linalg.norm(res.x - x_true) <= 1e-7 * np.linalg.norm(x_true)


def test_residual_is_orthogonal_to_the_atom_just_used():
    """(3) right after updating with atom i (unit columns): <r', psi_i> = c (1 - ||psi_i||^2) ~ 0."""
    psi_t, _, _, y = _random_problem(4)
    for T in (1, 2, 5, 9):
        res = oracle.mp(psi_t, y, 0.0, T)
        i = res.idx[-1]
        assert abs(float(res.r @ psi_t[i])) <= 1e-14 * np.linalg.norm(y)


def test_each_pick_is_the_brute_force_argmax_of_the_current_residual():
    """Replays the run step by step in numpy: at every t the chosen atom is argmax |Psi^T r_t|."""
    psi_t, _, _, y = _random_problem(5, N=24, M=16, K=3)
    res = oracle.mp(psi_t, y, 1e-6, 60)
    r = y.copy()
    for t in range(res.n_iter):
        c = psi_t @ r
        best = np.max(np.abs(c))
        i = min(m for m in range(len(c)) if abs(c[m]) == best)
        assert res.idx[t] == i
        assert res.c[t] == pytest.approx(c[i], rel=1e-12, abs=1e-15)
        r = r - c[i] * psi_t[i]


# ----------------------------------------------------------------------------- symmetries
def test_scaling_permutation_negation_symmetries():
    psi_t, _, _, y = _random_problem(6)
    base = oracle.mp(psi_t, y, 1e-8, 300)
    # scaling y by a power of two scales x~, r exactly, same indices and n_iter
    sc = oracle.mp(psi_t, 8.0 * y, 1e-8, 300)
    assert sc.n_iter == base.n_iter and np.array_equal(sc.idx, base.idx)
    assert np.array_equal(sc.x, 8.0 * base.x) and np.array_equal(sc.r, 8.0 * base.r)
    # permuting atoms permutes x~ (no exact ties in a random instance)
    perm = np.random.default_rng(0).permutation(psi_t.shape[0])
    pr = oracle.mp(np.ascontiguousarray(psi_t[perm]), y, 1e-8, 300)
    assert pr.n_iter == base.n_iter and np.array_equal(perm[pr.idx], base.idx)
    assert np.array_equal(pr.x, base.x[perm])
    # negating one atom negates its coefficient only
    j = int(base.idx[0])
    neg = psi_t.copy(); neg[j] = -neg[j]
    ng = oracle.mp(neg, y, 1e-8, 300)
    flip = np.ones(psi_t.shape[0]); flip[j] = -1.0
    assert np.array_equal(ng.idx, base.idx) and np.array_equal(ng.x, flip * base.x)
    assert np.array_equal(ng.r, base.r)


# ----------------------------------------------------------------------------- edge cases
def test_edge_cases():
    psi_t, _, _, y = _random_problem(8)
    M, N = psi_t.shape
    z = oracle.mp(psi_t, np.zeros(N), 1e-5, 10)          # y = 0: 0 > eps*0 is false
    assert z.n_iter == 0 and not z.x.any() and not z.r.any()
    m0 = oracle.mp(psi_t, y, 1e-5, 0)                     # T = 0
    assert m0.n_iter == 0 and not m0.x.any() and np.array_equal(m0.r, y)
    e0 = oracle.mp(psi_t, y, 0.0, 37)                     # eps = 0: runs to T
    assert e0.n_iter == 37
    e1 = oracle.mp(psi_t, y, 1.0, 37)                     # eps >= 1: ||y|| > ||y|| false
    assert e1.n_iter == 0
    with pytest.raises(ValueError):
        oracle.mp(psi_t, y, -1.0, 3)


def test_orthogonal_residual_runs_to_T_with_noop_updates():
    """max|c| = 0 while ||r|| > eps||y||: the paper's loop makes no-op updates until t = T."""
    psi_t = np.zeros((2, 3)); psi_t[0, 0] = 1.0; psi_t[1, 1] = 1.0
    y = np.array([0.0, 0.0, 2.0])
    res = oracle.mp(psi_t, y, 1e-3, 5)
    assert res.n_iter == 5 and list(res.idx) == [0] * 5 and not res.x.any() and np.array_equal(res.r, y)


# ----------------------------------------------------------------------------- normalisation (Eq. 4)
def test_normalize_columns():
    raw = synth.gaussian_dictionary(40, 30, 9).astype(np.float64)
    raw[7] = 0.0                                            # zero column stays zero
    out, norms = oracle.normalize_columns(raw)
    np.testing.assert_allclose(norms, np.linalg.norm(raw, axis=1), rtol=1e-15)
    nn = np.linalg.norm(out, axis=1)
    assert nn[7] == 0.0 and norms[7] == 0.0
    np.testing.assert_allclose(np.delete(nn, 7), 1.0, atol=4e-16)
    again, n2 = oracle.normalize_columns(out)              # idempotent to rounding
    np.testing.assert_allclose(again, out, atol=3e-16)
    # direction preserved, not just length
    np.testing.assert_allclose(out[3] * norms[3], raw[3], rtol=1e-15)
    # Bernoulli +-1/sqrt(N), N a power of 4: columns exactly unit, returned unchanged (Eq. 13)
    bern = synth.bernoulli_dictionary(64, 10, 1).astype(np.float64)
    assert set(np.unique(bern)) == {-0.125, 0.125}
    b2, bn = oracle.normalize_columns(bern)
    assert np.array_equal(b2, bern) and np.all(bn == 1.0)


# ----------------------------------------------------------------------------- the two instantiations, replay, batched, Eq. 14
def test_f32_instantiation_promotes_exactly():
    psi32, _, _, y = _random_problem(10, dtype=np.float32)
    a = oracle.mp(psi32, y, 1e-7, 200)
    b = oracle.mp(psi32.astype(np.float64), y, 1e-7, 200)
    assert a.n_iter == b.n_iter and np.array_equal(a.idx, b.idx)
    assert np.array_equal(a.x, b.x) and np.array_equal(a.r, b.r) and np.array_equal(a.gap, b.gap)


def test_padded_leading_dimension_is_honoured():
    """ld > N: rows are read with stride ld and the padding (NaN here) is never touched."""
    psi_t, _, _, y = _random_problem(15)
    M, N = psi_t.shape
    for dtype in (np.float64, np.float32):
        wide = np.full((M, N + 8), np.nan, dtype=dtype)
        wide[:, :N] = psi_t
        a = oracle.mp(wide[:, :N], y, 1e-6, 200)
        b = oracle.mp(np.ascontiguousarray(wide[:, :N]), y, 1e-6, 200)
        assert a.n_iter == b.n_iter > 0 and np.array_equal(a.idx, b.idx)
        assert np.array_equal(a.x, b.x) and np.array_equal(a.r, b.r)
        rp = oracle.mp_replay(wide[:, :N], y, a.idx, a.c)
        assert np.array_equal(rp.x, a.x) and np.array_equal(rp.argmax_ref, a.idx)
        np.testing.assert_array_equal(oracle.correlate(wide[:, :N], y), oracle.correlate(np.ascontiguousarray(wide[:, :N]), y))


def test_replay_along_own_trace_reproduces_the_run():
    psi_t, _, _, y = _random_problem(12)
    run = oracle.mp(psi_t, y, 1e-8, 300)
    for c_run in (None, run.c):
        rp = oracle.mp_replay(psi_t, y, run.idx, c_run)
        assert np.array_equal(rp.argmax_ref, run.idx)
        assert np.array_equal(rp.c_at_idx, run.c) and np.array_equal(rp.cmax_ref, np.abs(run.c))
        assert np.array_equal(rp.x, run.x) and np.array_equal(rp.r, run.r)
        assert np.array_equal(rp.rnorm, run.rnorm) and np.array_equal(rp.gap, run.gap)


def test_replay_with_imposed_atoms_and_steps_holds_y_minus_psi_x():
    """Forcing (idx, step) keeps the oracle state at exactly y - sum_t step_t psi_idx_t."""
    psi_t, _, _, y = _random_problem(13)
    rng = np.random.default_rng(1)
    idx = rng.integers(0, psi_t.shape[0], 25).astype(np.int32)
    steps = rng.standard_normal(25)
    rp = oracle.mp_replay(psi_t, y, idx, steps)
    x = np.zeros(psi_t.shape[0]); np.add.at(x, idx, steps)
    np.testing.assert_allclose(rp.x, x, atol=1e-14)
    np.testing.assert_allclose(rp.r, y - psi_t.T @ x, atol=1e-13)
    # the recorded reference quantities are those of the state BEFORE each forced step
    r = y.copy()
    for t in range(25):
        c = psi_t @ r
        assert rp.argmax_ref[t] == int(np.argmax(np.abs(c)))
        assert rp.c_at_idx[t] == pytest.approx(c[idx[t]], rel=1e-12, abs=1e-14)
        top = np.sort(np.abs(c))[-2:]
        assert rp.gap[t] == pytest.approx((top[1] - top[0]) / top[1], rel=1e-9, abs=1e-14)
        r = r - steps[t] * psi_t[idx[t]]


def test_batched_equals_independent_runs():
    psi32, _, _, _ = _random_problem(14, dtype=np.float32)
    M, N = psi32.shape
    Y = np.stack([synth.encode(psi32, *synth.sparse_signal(M, 5, 14, "normal", signal=b)) for b in range(4)])
    Y[2] = 0.0
    X, R, n_iter = oracle.mp_batched(psi32, Y, 1e-6, 200)
    for b in range(4):
        one = oracle.mp(psi32, Y[b], 1e-6, 200)
        assert n_iter[b] == one.n_iter and np.array_equal(X[b], one.x) and np.array_equal(R[b], one.r)
    assert n_iter[2] == 0 and len(set(n_iter.tolist())) > 1


def test_reconstruction_error_eq14():
    """Eq. 14 on a hand-computed example: (0.1^2 + 0.1^2)/1 * 100 = 2 %."""
    assert oracle.reconstruction_error_pct([0.9, 0.1, 0.0], [1.0, 0.0, 0.0]) == pytest.approx(2.0, rel=1e-12)
    assert oracle.reconstruction_error_pct([1.0, 2.0], [1.0, 2.0]) == 0.0


# ----------------------------------------------------------------------------- the paper's own (prose) claims
def _golden():
    out = {}
    with open(os.path.join(GOLDEN, "paper_claims.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = [s.strip() for s in line.split("=")]
                out[k] = v
    return out


@pytest.mark.parametrize("M,seed", [(600, 1), (1000, 2)])
def test_paper_sweep_parameters_finish_within_T_and_recover_x(M, seed):
    """with sigma=0.07, rho=0.5, eps=1e-7, T=N, Bernoulli Psi, U[-1,1] nonzeros, 'the MP
    algorithm is able to find the solution with an error eps in maximum N iteration steps' -- under
    the listings' threshold sqrt(eps*||y||) (A1 P:272-275).  And P:106: exact recovery (Eq. 14 -> 0 %)."""
    g = _golden()
    K = int(float(g["sweep_sigma"]) * M)
    N = int(float(g["sweep_rho"]) * M)
    eps = float(g["sweep_eps"])
    T = int(g["sweep_T_over_N"]) * N
    assert g["sweep_dictionary"] == "bernoulli" and g["sweep_values"] == "uniform"
    psi_t = synth.bernoulli_dictionary(N, M, seed)
    x, S = synth.sparse_signal(M, K, seed, "uniform")
    y = synth.encode(psi_t, x, S).astype(np.float64)
    ny = np.linalg.norm(y)
    eps_listing = math.sqrt(eps * ny) / ny                  # same threshold expressed as a fraction of ||y||
    res = oracle.mp(psi_t, y, eps_listing, T)
    assert res.n_iter < T                                   # claim_done_within_T
    assert oracle.reconstruction_error_pct(res.x, x) < 1e-3
    full = oracle.mp(psi_t, y, 0.0, T)                      # exactly T = N steps
    assert oracle.reconstruction_error_pct(full.x, x) < 1e-5   # "recovers exactly"


# ----------------------------------------------------------------------------- Eq. 2 (encode), the step before the path
def test_encode_sparse_pins():
    """Eq. 2, y = Psi x for a K-sparse x: a unit coefficient returns the atom itself; the result equals numpy's
    float64 dense product Psi^T-major @ x to rounding; a brute-force Python double loop on a tiny case is matched exactly;
    repeated indices accumulate (A2 P:328-332 draws the support with replacement); power-of-two scaling is exact."""
    rng = np.random.default_rng(3)
    M, N, K = 40, 12, 5
    psi = rng.standard_normal((M, N)).astype(np.float32)
    for m in (0, 7, M - 1):
        assert np.array_equal(oracle.encode_sparse(psi, [m], [1.0]), psi[m].astype(np.float64))
    idx = rng.choice(M, K, replace=False); val = rng.standard_normal(K)
    y = oracle.encode_sparse(psi, idx, val)
    x = np.zeros(M); x[idx] = val
    dense = psi.astype(np.float64).T @ x
    assert np.allclose(y, dense, rtol=0, atol=1e-15 * np.abs(psi).max() * np.abs(val).sum())
    brute = [sum(float(val[k]) * float(psi[idx[k], n]) for k in range(K)) for n in range(N)]
    acc = []
    for n in range(N):                                   # the same ascending-k order, one add at a time
        s = 0.0
        for k in range(K):
            s += float(val[k]) * float(psi[idx[k], n])
        acc.append(s)
    assert list(y) == acc and np.allclose(y, brute, atol=1e-15)
    assert np.array_equal(oracle.encode_sparse(psi, [3, 3], [0.5, 0.25]), 0.75 * psi[3].astype(np.float64))
    assert np.array_equal(oracle.encode_sparse(psi, idx, 4.0 * val), 4.0 * y)
    assert np.array_equal(oracle.encode_sparse(psi, [], []), np.zeros(N))
    with pytest.raises(ValueError):
        oracle.encode_sparse(psi, [M], [1.0])
    # and it agrees with the input generator's encode (which bench.py and the parity tests use to make y)
    from paper_0809_1833_b200 import synth
    assert np.array_equal(y.astype(np.float32), synth.encode(psi, x, np.sort(idx))) or \
        np.allclose(y.astype(np.float32), synth.encode(psi, x, np.sort(idx)), rtol=2e-7)


# ----------------------------------------------------------------------------- Orthogonal MP
def _unit_rows(rng, M, N):
    p = rng.standard_normal((M, N))
    return (p / np.linalg.norm(p, axis=1, keepdims=True)).astype(np.float32)


def test_omp_least_squares_and_orthogonality():
    """After every step the coefficients are the least-squares solution on the selected atoms: they equal numpy's lstsq,
    the residual is orthogonal to every selected atom, no atom is taken twice, ||r|| is non-increasing, and a K-sparse x
    in the exact-recovery regime is recovered in exactly K steps (each step removes one atom for good)."""
    rng = np.random.default_rng(11)
    M, N, K = 300, 80, 7
    psi = _unit_rows(rng, M, N)
    P = psi.astype(np.float64)
    s = rng.choice(M, K, replace=False)
    x = np.zeros(M); x[s] = rng.standard_normal(K) + np.sign(rng.standard_normal(K))
    y = P.T @ x
    res = oracle.omp(psi, y, 1e-12, 40)
    assert res.status == 0 and res.n_iter == K and set(res.idx.tolist()) == set(s.tolist())
    assert len(set(res.idx.tolist())) == K and np.all(np.diff(res.rnorm) <= 1e-15)
    assert np.allclose(res.x, x, atol=1e-13) and res.rnorm[-1] <= 1e-13 * res.rnorm[0]
    for t in range(1, K + 1):                                               # every prefix is a least-squares fit
        rp = oracle.omp(psi, y, 0.0, 0, idx_force=res.idx[:t])
        S = res.idx[:t]
        z = np.linalg.lstsq(P[S].T, y, rcond=None)[0]
        assert np.allclose(rp.x[S], z, atol=1e-12) and not np.any(np.delete(rp.x, S))
        assert np.max(np.abs(P[S] @ rp.r)) <= 1e-13 * np.linalg.norm(y)
        assert np.allclose(rp.r, y - P[S].T @ z, atol=1e-12)


def test_omp_equals_mp_on_orthonormal_dictionary_and_first_step():
    """Orthonormal Psi: the refit changes nothing, OMP = MP (same atoms, same coefficients).  Any Psi: the first OMP step is
    the first MP step divided by ||psi_i||^2 (= 1 for unit atoms)."""
    N = 64
    H = np.array([[1.0]])
    while H.shape[0] < N:
        H = np.block([[H, H], [H, -H]])
    psi = (H / 8.0).astype(np.float32)
    rng = np.random.default_rng(2)
    s = rng.choice(N, 6, replace=False); x = np.zeros(N); x[s] = rng.standard_normal(6)
    y = psi.astype(np.float64).T @ x
    a = oracle.omp(psi, y, 1e-12, 30); b = oracle.mp(psi, y, 1e-12, 30)
    assert a.n_iter == b.n_iter == 6 and np.array_equal(a.idx, b.idx) and np.allclose(a.x, b.x, atol=1e-15)
    psi2 = _unit_rows(rng, 50, 20); y2 = rng.standard_normal(20)
    a1 = oracle.omp(psi2, y2, 0.0, 1); b1 = oracle.mp(psi2, y2, 0.0, 1)
    i = int(a1.idx[0])
    assert i == int(b1.idx[0]) and a1.gap[0] == b1.gap[0]
    nrm2 = float(np.sum(psi2[i].astype(np.float64) ** 2))
    assert abs(a1.x[i] - b1.x[i] / nrm2) <= 1e-15


def test_omp_two_atom_closed_form_and_edge_cases():
    """Two atoms with coherence mu, y in their span: MP needs infinitely many steps (||r|| shrinks by |mu| each), OMP is exact
    after two.  y = 0, T = 0, eps >= 1 give 0 steps; T is capped at N; a forced repeated atom ends the run (status 2)."""
    mu = 0.9
    psi = np.zeros((2, 4), np.float32); psi[0, 0] = 1.0; psi[1, 0] = mu; psi[1, 1] = np.sqrt(1 - np.float64(mu) ** 2)
    P = psi.astype(np.float64)
    y = 2.0 * P[0] - 1.5 * P[1]
    res = oracle.omp(psi, y, 1e-13, 10)
    assert res.n_iter == 2 and np.allclose(res.x, [2.0, -1.5], atol=1e-7) and res.rnorm[-1] <= 1e-7
    assert oracle.mp(psi, y, 1e-6, 1000).n_iter > 50
    assert oracle.omp(psi, np.zeros(4), 1e-5, 10).n_iter == 0
    assert oracle.omp(psi, y, 1e-5, 0).n_iter == 0 and oracle.omp(psi, y, 1.0, 10).n_iter == 0
    rng = np.random.default_rng(4)
    psi3 = _unit_rows(rng, 40, 6)
    assert oracle.omp(psi3, rng.standard_normal(6), 0.0, 100).n_iter <= 6
    dup = oracle.omp(psi3, rng.standard_normal(6), 0.0, 0, idx_force=[3, 5, 3])
    assert dup.status == 2 and dup.n_iter == 2


def test_rowmajor_ingestion_is_the_index_swap_and_keeps_the_method():
    """atom_major_from_rowmajor: psi_t[m, n] = Psi[n, m] checked index by index, and MP on the converted dictionary equals a
    numpy gemv/argmax/axpy loop run directly on the paper's row-major array (A2 P:464-471 in that layout)."""
    rng = np.random.default_rng(21)
    N, M = 7, 11
    psi = rng.standard_normal((N, M))
    psi /= np.linalg.norm(psi, axis=0, keepdims=True)
    pt = oracle.atom_major_from_rowmajor(psi)
    assert pt.shape == (M, N) and all(pt[m, n] == psi[n, m] for m in range(M) for n in range(N))
    x = np.zeros(M); x[[2, 9]] = [1.5, -0.7]
    y = psi @ x
    res = oracle.mp(pt, y, 0.0, 6)
    r = y.copy(); xs = np.zeros(M)
    for t in range(6):
        c = psi.T @ r                                   # gemv on the row-major array
        i = int(np.argmax(np.abs(c)))                   # first occurrence = lowest index
        xs[i] += c[i]; r = r - c[i] * psi[:, i]         # axpy with the stride-M column
        assert res.idx[t] == i
    assert np.allclose(res.x, xs, atol=1e-14) and np.allclose(res.r, r, atol=1e-14)
