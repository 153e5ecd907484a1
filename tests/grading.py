"""Grading of a GPU Matching Pursuit run against the CPU oracle (test infrastructure).

Implements the parity contract of BASELINE.json's north_star under the readings listed in DESIGN.md:

  G1 free-running: the GPU index sequence equals the oracle's up to the first iteration whose top-two
     relative gap of |c| (on the oracle's own state) is <= 1e-4 plus the drift allowance
     (|<d, psi_ref>| + |<d, psi_gpu>|) / max|c|, d = the difference of the two residuals accumulated from the
     step-value errors so far (each bounded by G3); the Grade records whether and how much of it was used
     -- after a legal near-tie flip the two runs are different trajectories and cannot be compared step by step.
  G2 teacher-forced replay over the WHOLE GPU trace: the oracle is advanced with the GPU's own (index,
     step) pairs, so its state is the exact-arithmetic image of the GPU state; at every iteration the
     GPU's pick must be the oracle's argmax, or a near-tie (gap <= 1e-4 and |c_ref[pick]| >= (1-1e-4) max).
  G3 every step value: |c_gpu - c_ref[pick]| <= C_TOL * ||r_t||  (fp32 dot product of N terms against a
     float64 reference; bound derived in DESIGN.md "Tolerances").
  G4 final residual: | ||r_gpu|| - ||r_replay|| | <= 1e-4 ||r_replay||  (north_star) -- and, tighter,
     the vector itself to fp32 rounding;  x_gpu equals the replay's x to fp32 rounding.
  G5 stop rule: the GPU continued exactly while ||r|| > eps ||y|| and t < T, judged on the replay's norms.
  G6 exact-recovery regime (oracle stops by eps with ||x_ref - x_true|| <= 1e-4 ||x_true||): selected atoms
     == true support, ||x_gpu - x_ref|| <= 1e-4 ||x_ref||.
"""
from __future__ import annotations

import dataclasses

import numpy as np

import oracle

GAP_TOL = 1e-4      # north_star: "top-two |c| gap exceeds 1e-4 relative"
C_TOL = 4e-6        # |c_gpu - c_ref| / ||r_t||, see DESIGN.md "Tolerances"


def c_tol_tensor_core(N: int) -> float:
    """Step-value tolerance of the batched tensor-core path: the tcgen05 fp32 accumulator is
    truncated (not rounded) on every UMMA, at most one ulp = 2^-23 of the running sum (|running sum| <= ||r||), and
    each split-K accumulator chain is N/32 UMMAs long; measured bias is about 0.37 of this bound."""
    return C_TOL + (N / 32.0) * 2.0 ** -23
NORM_TOL = 1e-4     # north_star: final ||r|| within 1e-4 relative
X_TOL = 1e-4        # north_star: ||x_gpu - x_ref|| / ||x_ref||

# Caps on the two state-drift allowances (readings R14b, R16b), so that neither can grow without anybody noticing:
#   * the drift itself is bounded by what G3 tolerates: d_{s+1} = (I - psi_s psi_s^T) d_s + e_s psi_s with e_s = c_gpu,s - <r_image,s, psi_s>
#     (the oracle's free-running step is its own correlation, which already contains <d_s, psi_s>), a projection is non-expansive,
#     hence ||d|| <= sum_s |e_s| <= sum_s c_tol ||r_s||.  Asserted below on the replay's norms, after G3.
#   * ceilings with about 2x headroom over the worst case of the full GPU session (1425 grades: G1 allowance used 33 times, largest
#     8.3e-3 at an oracle gap of 7.1e-3; n_iter drift used once, 1.2e-3 of the threshold).  Beyond them a run is looked at by hand.
#   * the session as a whole may use them at most G1_ALLOWANCE_MAX_USES / N_ITER_DRIFT_MAX_USES times (tests/conftest.py).
G1_ALLOWANCE_CEILING = 2e-2
N_ITER_DRIFT_CEILING = 5e-3        # ||d|| / (eps ||y||)
G1_ALLOWANCE_MAX_USES = 50
N_ITER_DRIFT_MAX_USES = 3

# Every grade of the session, so that the use of the G1 allowance and the worst observed errors are visible
# (tests/conftest.py prints the summary and writes it to gpurun_out/grading_summary.json when that folder exists).
LOG: list[dict] = []


@dataclasses.dataclass
class Grade:
    n_iter_gpu: int
    n_iter_ref: int
    first_divergence: int          # -1 if the free-running sequences agree on their common prefix
    near_ties: int                 # iterations with gap <= GAP_TOL (replay)
    flips: int                     # iterations where the GPU pick != oracle argmax (all legal if we got here)
    max_c_err: float               # max |c_gpu - c_ref| / ||r_t||
    rnorm_rel_err: float
    x_rel_err_vs_ref: float
    exact_recovery: bool
    g1_allowance_used: bool = False    # the free-running sequences diverged at an oracle gap ABOVE GAP_TOL, accepted by R14b
    g1_allowance: float = 0.0          # 2 ||d|| / max|c| at that divergence (0 if the sequences never diverged)
    g1_gap: float = 0.0                # the oracle's top-two gap at that divergence
    n_iter_drift_used: bool = False    # n_iter differs by one on identical sequences, edge outside NORM_TOL, accepted by R16b
    n_iter_drift: float = 0.0          # ||d|| / (eps ||y||) at that edge (0 if n_iter agreed)


def grade_single(psi32: np.ndarray, y32: np.ndarray, eps: float, max_iter: int,
                 x_gpu, r_gpu, n_iter_gpu, idx_gpu, c_gpu, *, x_true=None, support=None,
                 nthreads: int | None = None, ref: "oracle.MPResult | None" = None, c_tol: float = C_TOL) -> Grade:
    nthreads = nthreads or oracle.default_threads()
    eps = float(np.float32(eps))                       # the very float the GPU received
    y = y32.astype(np.float64)
    t_gpu = int(n_iter_gpu)
    idx_gpu = np.asarray(idx_gpu[:t_gpu], dtype=np.int32)
    c_gpu = np.asarray(c_gpu[:t_gpu], dtype=np.float64)
    x_gpu = np.asarray(x_gpu, dtype=np.float64)
    r_gpu = np.asarray(r_gpu, dtype=np.float64)
    M, N = psi32.shape
    assert 0 <= t_gpu <= max_iter
    assert np.all((idx_gpu >= 0) & (idx_gpu < M)), "index out of range"

    if ref is None:
        ref = oracle.mp(psi32, y, eps, max_iter, nthreads)
    ny = ref.rnorm[0] if ref.rnorm.size else 0.0

    # ---- G1 free-running ------------------------------------------------------------------------------
    L = min(t_gpu, ref.n_iter)
    diff = np.nonzero(idx_gpu[:L] != ref.idx[:L])[0]
    first_div = int(diff[0]) if diff.size else -1
    g1_used, g1_allow, g1_gap = False, 0.0, 0.0
    if first_div >= 0:
        # The oracle's gap is measured on the ORACLE's state; the GPU decided on ITS state.  Up to first_div both
        # took the same atoms, so the two residuals differ only by the accumulated step-value errors (each within
        # C_TOL ||r_s||, G3): d = sum_s (c_gpu,s - c_ref,s) psi_idx_s.  Every correlation then differs by at most
        # ||d|| (unit atoms), which moves the top-two comparison by at most 2 ||d|| / max|c|.  A divergence is legal
        # if the oracle's gap is within GAP_TOL plus that drift allowance; G2 below still requires the GPU's pick
        # to be the argmax (or a <= 1e-4 near-tie) of the exact-arithmetic image of its own state at EVERY step.
        # The allowance is the EXACT shift of the two correlations involved, |<d, psi_ref>| + |<d, psi_gpu>| (not the bound
        # 2 ||d||), so it is as small as the accumulated step errors allow.  No constant cap can be derived for it: late in a
        # run ||r_t|| has fallen by 4-5 orders of magnitude while d carries the (tolerated, G3) step errors of the early,
        # large iterations, so the two runs are then simply two different valid trajectories.  Its use and size are
        # recorded in the Grade and summarised at the end of the session (tests/conftest.py).
        d = np.zeros(N)
        for s_ in range(first_div):
            d += (c_gpu[s_] - ref.c[s_]) * psi32[idx_gpu[s_]].astype(np.float64)
        cmax = abs(ref.c[first_div])
        shift = abs(float(d @ psi32[ref.idx[first_div]].astype(np.float64))) + abs(float(d @ psi32[idx_gpu[first_div]].astype(np.float64)))
        g1_allow = shift / max(cmax, np.finfo(np.float64).tiny)
        g1_gap = float(ref.gap[first_div])
        g1_used = bool(g1_gap > GAP_TOL)
        allowance = GAP_TOL + g1_allow
        g1_drift = float(np.linalg.norm(d))
        assert not g1_used or g1_allow <= G1_ALLOWANCE_CEILING, (
            f"free-running divergence at t={first_div} needs a state-drift allowance of {g1_allow:.3e} > ceiling {G1_ALLOWANCE_CEILING} "
            f"(oracle gap {g1_gap:.3e}): the step errors have grown, look at G3's margins")
        assert ref.gap[first_div] <= allowance, (
            f"free-running sequences diverge at t={first_div} where the oracle's top-two gap is {ref.gap[first_div]:.3e} "
            f"> {GAP_TOL} + state-drift allowance {allowance - GAP_TOL:.3e}")

    # ---- G2/G3 teacher-forced replay ------------------------------------------------------------------------
    rp = oracle.mp_replay(psi32, y, idx_gpu, c_gpu, nthreads)
    same = idx_gpu == rp.argmax_ref
    legal = same | ((rp.gap <= GAP_TOL) & (np.abs(rp.c_at_idx) >= (1.0 - GAP_TOL) * rp.cmax_ref))
    bad = np.nonzero(~legal)[0]
    assert bad.size == 0, (
        f"{bad.size} illegal picks, first at t={bad[0]}: gpu idx {idx_gpu[bad[0]]} |c_ref|={abs(rp.c_at_idx[bad[0]]):.9e} "
        f"vs oracle idx {rp.argmax_ref[bad[0]]} max={rp.cmax_ref[bad[0]]:.9e} gap={rp.gap[bad[0]]:.3e}")
    c_err = np.abs(c_gpu - rp.c_at_idx) / np.maximum(rp.rnorm[:t_gpu], np.finfo(np.float64).tiny) if t_gpu else np.zeros(0)
    max_c_err = float(c_err.max()) if t_gpu else 0.0
    assert max_c_err <= c_tol, f"step value error {max_c_err:.3e} ||r|| at t={int(c_err.argmax())} exceeds {c_tol}"
    if first_div >= 0:                                     # the drift G1 allowed for is within what G3 tolerates (see the caps above)
        bound = c_tol * float(np.sum(rp.rnorm[:first_div]))
        assert g1_drift <= bound * (1.0 + 1e-6) + 1e-300, f"state drift ||d|| = {g1_drift:.3e} exceeds the G3-derived bound {bound:.3e}"

    # ---- G4 final residual and coefficients ---------------------------------------------------------------------
    nr_gpu = float(np.linalg.norm(r_gpu))
    nr_rep = float(rp.rnorm[t_gpu])
    rn_err = abs(nr_gpu - nr_rep) / nr_rep if nr_rep > 0 else abs(nr_gpu)
    assert rn_err <= NORM_TOL, f"final ||r|| off by {rn_err:.3e} relative"
    assert np.linalg.norm(r_gpu - rp.r) <= 1.2e-7 * np.linalg.norm(rp.r) + 1e-30, "r is not the fp32 rounding of y - Psi x~"
    assert np.all(np.abs(x_gpu - rp.x) <= 6e-8 * np.abs(rp.x) + 1e-45), "x is not the fp32 rounding of the accumulated steps"

    # ---- G5 stop rule ------------------------------------------------------------------------------------------------
    thr = eps * ny
    if t_gpu:
        assert np.all(rp.rnorm[:t_gpu] > thr * (1.0 - 1e-9)), "GPU continued although ||r|| <= eps ||y||"
    if t_gpu < max_iter:
        assert rp.rnorm[t_gpu] <= thr * (1.0 + 1e-9), "GPU stopped although ||r|| > eps ||y|| and t < T"

    # ---- n_iter --------------------------------------------------------------------------------------------------------
    nd_used, nd_rel = False, 0.0
    if first_div < 0:
        if t_gpu != ref.n_iter:
            # Only a tie at the stopping threshold may move n_iter by one (R16).  The oracle's ||r|| is measured on the ORACLE's
            # state; the GPU stopped (G5 above, strict) on ITS state.  Both took the same atoms, so the two residuals differ by
            # d = sum_s (c_gpu,s - c_ref,s) psi_idx_s (every term within G3), and the two norms at the edge by at most ||d||
            # (triangle inequality) -- the same state drift G1 allows for (R14b), applied to the stop test (R16b).  Late in a
            # run ||r|| = eps ||y|| is 1e-5 ||y|| while d carries the tolerated step errors of the early iterations
            # (<= C_TOL ||r_s|| each), so ||d|| can exceed NORM_TOL * thr; its use and size are recorded in the Grade.
            assert abs(t_gpu - ref.n_iter) == 1, f"n_iter {t_gpu} vs oracle {ref.n_iter} on identical sequences"
            e = min(t_gpu, ref.n_iter)
            edge = ref.rnorm[e]
            d = np.zeros(N)
            for s_ in range(e):
                d += (c_gpu[s_] - ref.c[s_]) * psi32[idx_gpu[s_]].astype(np.float64)
            nd = float(np.linalg.norm(d))
            nd_rel = nd / thr if thr > 0 else 0.0
            nd_used = bool(abs(edge - thr) > NORM_TOL * thr)
            bound = c_tol * float(np.sum(rp.rnorm[:e]))
            assert nd <= bound * (1.0 + 1e-6) + 1e-300, f"state drift ||d|| = {nd:.3e} exceeds the G3-derived bound {bound:.3e}"
            assert not nd_used or nd_rel <= N_ITER_DRIFT_CEILING, (
                f"n_iter differs by one with a state drift of {nd_rel:.3e} of the threshold > ceiling {N_ITER_DRIFT_CEILING}")
            assert abs(edge - thr) <= NORM_TOL * thr + nd, (
                f"n_iter differs by one away from the stopping threshold: | ||r_ref|| - thr | = {abs(edge - thr):.3e}, "
                f"NORM_TOL * thr = {NORM_TOL * thr:.3e}, state drift ||d|| = {nd:.3e}")

    # ---- G6 exact-recovery regime -----------------------------------------------------------------------------------------
    x_err_ref = float(np.linalg.norm(x_gpu - ref.x) / max(np.linalg.norm(ref.x), 1e-300)) if ref.n_iter else 0.0
    exact = False
    if x_true is not None and ref.n_iter < max_iter and np.linalg.norm(ref.x - x_true) <= X_TOL * np.linalg.norm(x_true):
        exact = True
        assert x_err_ref <= X_TOL, f"||x_gpu - x_ref||/||x_ref|| = {x_err_ref:.3e}"
        assert t_gpu < max_iter and np.linalg.norm(r_gpu) <= thr * (1 + 1e-6)
        if support is not None:
            sup = set(int(s) for s in support)
            if set(ref.idx.tolist()) == sup:           # strict form holds for the oracle -> must hold for the GPU
                assert set(idx_gpu.tolist()) == sup, "selected atoms differ from the true support"
            tau = 1e-3 * np.max(np.abs(x_true))
            off = np.ones(M, bool); off[list(sup)] = False
            assert not np.any(np.abs(x_gpu[off]) > tau), "off-support coefficient above tau"
            big = [m for m in sup if abs(x_true[m]) >= 2 * tau]
            assert np.all(np.abs(x_gpu[big]) > tau), "a true coefficient is missing"
    g = Grade(t_gpu, ref.n_iter, first_div, int(np.sum(rp.gap <= GAP_TOL)), int(np.sum(~same)),
              max_c_err, rn_err, x_err_ref, exact, g1_used, g1_allow, g1_gap, nd_used, nd_rel)
    LOG.append({"N": int(N), "M": int(M), "c_tol": float(c_tol), **dataclasses.asdict(g)})
    return g


def residual_at(psi32: np.ndarray, y32: np.ndarray, idx, c, t: int) -> np.ndarray:
    """y - sum_{s<t} c_s psi_{idx_s} in float64: the exact-arithmetic image of the run's state before step t."""
    r = y32.astype(np.float64).copy()
    idx = np.asarray(idx[:t]); c = np.asarray(c[:t], dtype=np.float64)
    if t:
        coef = np.zeros(psi32.shape[0]); np.add.at(coef, idx, c)
        for m in np.nonzero(coef)[0]:
            r -= coef[m] * psi32[m].astype(np.float64)
    return r


def grade_sampled(psi32, y32, idx_gpu, c_gpu, n_iter_gpu, r_gpu, sample_ts, nthreads=None, c_tol: float = C_TOL):
    """Full-size check on SAMPLED iterations the oracle can compute one by one: for each t in sample_ts the
    state is rebuilt in float64 from the GPU trace, one oracle correlation pass gives c_ref, and the GPU's pick
    and step must satisfy G2/G3.  Also checks the final residual (G4)."""
    nthreads = nthreads or oracle.default_threads()
    t_gpu = int(n_iter_gpu)
    out = []
    for t in sample_ts:
        if not 0 <= t < t_gpu:
            continue
        r = residual_at(psi32, y32, idx_gpu, c_gpu, t)
        c = oracle.correlate(psi32, r, nthreads)
        i_ref = oracle.argmax_abs(c)
        a = np.abs(c); a1 = a[i_ref]
        a2 = np.max(np.delete(a, i_ref)) if a.size > 1 else 0.0
        gap = (a1 - a2) / a1 if a1 > 0 else 0.0
        i = int(idx_gpu[t])
        assert i == i_ref or (gap <= GAP_TOL and a[i] >= (1 - GAP_TOL) * a1), f"illegal pick at sampled t={t}"
        err = abs(float(c_gpu[t]) - c[i]) / oracle.nrm2(r)
        assert err <= c_tol, f"step value error {err:.3e} at sampled t={t}"
        out.append((t, gap, err))
    r_fin = residual_at(psi32, y32, idx_gpu, c_gpu, t_gpu)
    nr = oracle.nrm2(r_fin)
    assert abs(np.linalg.norm(np.asarray(r_gpu, np.float64)) - nr) <= NORM_TOL * nr
    assert np.linalg.norm(np.asarray(r_gpu, np.float64) - r_fin) <= 1.2e-7 * nr + 1e-30
    return out
