"""Seeded synthetic inputs shaped like the paper's workloads (host side, numpy only).

This module is the ONE place both the CPU oracle's tests and the CUDA path's tests/bench
draw inputs from, so both sides see identical bits.  It holds none of the method's
arithmetic (no correlation, no argmax, no residual update, no normalisation): it only
draws random dictionaries and sparse signals and forms the measurement y = Psi x.

What the paper's workloads look like:
  * Psi is a random N x M matrix, Bernoulli +-1/sqrt(N) (Eq. 13) or Gaussian;
  * x is K-sparse with random support and random nonzeros (Eq. 1);
  * y = Psi x (Eq. 2);  N ~ c K log(M/K).
The paper seeds C rand() with time() (A1 P:238, A2 P:383) so nothing in it is
reproducible; we use a counter-based 64-bit hash instead (any element can be drawn
independently, chunk by chunk, in any order).

Layout: dictionaries are returned ATOM-MAJOR, psi_t[m, n] = Psi[n][m] (shape [M, N],
C-contiguous, float32) -- the layout the C-ABI library takes (include/mp_b200.h).
"""
from __future__ import annotations

import dataclasses
import os

import numpy as np

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(z: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on a uint64 array (wrapping arithmetic)."""
    z = (z + np.uint64(0x9E3779B97F4A7C15)) & _MASK
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _MASK
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _MASK
    return z ^ (z >> np.uint64(31))


def hash_u64(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Counter-based generator: 64 random bits for every (seed, stream, index)."""
    with np.errstate(over="ignore"):
        key = _mix64(np.asarray([seed & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))
        key = _mix64(key ^ np.uint64(stream & 0xFFFFFFFFFFFFFFFF))
        return _mix64(_mix64(np.asarray(index, dtype=np.uint64)) ^ key)


def uniform01(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """U(0,1) in float64, strictly inside (0,1): (top 53 bits + 0.5) / 2^53."""
    bits = hash_u64(seed, stream, index) >> np.uint64(11)
    return (bits.astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def standard_normal(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """N(0,1) in float64 by Box-Muller on two independent uniforms per index."""
    u1 = uniform01(seed, 2 * stream, index)
    u2 = uniform01(seed, 2 * stream + 1, index)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# stream ids (arbitrary, fixed)
_S_PSI, _S_SUPPORT, _S_VALUE, _S_SIGN = 1, 2, 3, 4
_CHUNK_ROWS_BYTES = 16 << 20


def _for_row_blocks(N: int, M: int, fill) -> None:
    """fill(m0, m1) over row blocks of the dictionary.  Every element is a function of (seed, stream, index) alone
    (counter-based), so the blocks are independent and are filled by a few threads (numpy releases the GIL)."""
    rows = max(1, _CHUNK_ROWS_BYTES // (8 * N))
    blocks = [(m0, min(M, m0 + rows)) for m0 in range(0, M, rows)]
    workers = min(len(blocks), os.cpu_count() or 1, 16)
    if workers <= 1:
        for b in blocks:
            fill(*b)
        return
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(workers) as ex:
        list(ex.map(lambda b: fill(*b), blocks))


def gaussian_dictionary(N: int, M: int, seed: int) -> np.ndarray:
    """psi_t[M, N] float32, entries i.i.d. N(0,1) (drawn in float64, rounded once).
    NOT normalised -- normalising columns (Eq. 4) is a step of the method."""
    out = np.empty((M, N), dtype=np.float32)

    def fill(m0, m1):
        idx = np.arange(m0 * N, m1 * N, dtype=np.uint64)
        out[m0:m1] = standard_normal(seed, _S_PSI, idx).reshape(m1 - m0, N).astype(np.float32)
    _for_row_blocks(N, M, fill)
    return out


def bernoulli_dictionary(N: int, M: int, seed: int) -> np.ndarray:
    """psi_t[M, N] float32, entries +-1/sqrt(N) equiprobable (Eq. 13).
    1/sqrt(N) is computed in float64 and rounded to float32 once (exact when N is a
    power of 4, e.g. N=4096 -> 1/64)."""
    a = np.float32(1.0 / np.sqrt(float(N)))
    out = np.empty((M, N), dtype=np.float32)

    def fill(m0, m1):
        idx = np.arange(m0 * N, m1 * N, dtype=np.uint64)
        bit = (hash_u64(seed, _S_PSI, idx) >> np.uint64(63)).astype(np.bool_)
        out[m0:m1] = np.where(bit, a, -a).reshape(m1 - m0, N)
    _for_row_blocks(N, M, fill)
    return out


def sparse_support(M: int, K: int, seed: int, signal: int = 0) -> np.ndarray:
    """K distinct indices uniform without replacement (partial Fisher-Yates driven by the
    hash), returned in draw order.  (The paper draws rand()%M WITH replacement,
    A2 P:328-332; BASELINE.json's configs say without.)"""
    if not 0 <= K <= M:
        raise ValueError("need 0 <= K <= M")
    u = uniform01(seed, _S_SUPPORT + 16 * signal, np.arange(K, dtype=np.uint64))
    perm: dict[int, int] = {}
    out = np.empty(K, dtype=np.int64)
    for k in range(K):
        j = k + int(u[k] * (M - k))
        vk, vj = perm.get(k, k), perm.get(j, j)
        perm[k], perm[j] = vj, vk
        out[k] = vj
    return out


def sparse_signal(M: int, K: int, seed: int, values: str = "normal", signal: int = 0):
    """K-sparse x in R^M (float64) and its support.
    values: 'normal'   -> N(0,1)                         (configs 1, 3, 4, 5)
            'pm_uniform' -> +-1 * U[0.5,1.5]             (config 2)
            'uniform'  -> U[-1,1]                        (the paper's own choice)"""
    S = sparse_support(M, K, seed, signal)
    k = np.arange(K, dtype=np.uint64)
    if values == "normal":
        v = standard_normal(seed, _S_VALUE + 16 * signal, k)
    elif values == "pm_uniform":
        mag = 0.5 + uniform01(seed, _S_VALUE + 16 * signal, k)
        sgn = np.where(hash_u64(seed, _S_SIGN + 16 * signal, k) >> np.uint64(63), 1.0, -1.0)
        v = sgn * mag
    elif values == "uniform":
        v = 2.0 * uniform01(seed, _S_VALUE + 16 * signal, k) - 1.0
    else:
        raise ValueError(values)
    x = np.zeros(M, dtype=np.float64)
    x[S] = v
    return x, S


def encode(psi_t: np.ndarray, x: np.ndarray, support: np.ndarray | None = None) -> np.ndarray:
    """Measurement y = Psi x (Eq. 2) in float64 from the given (fp32) dictionary
    bits, rounded to float32 once.  Only the support rows are touched (others multiply 0)."""
    if support is None:
        support = np.nonzero(x)[0]
    y = np.zeros(psi_t.shape[1], dtype=np.float64)
    for m in np.sort(np.asarray(support)):
        y += float(x[m]) * psi_t[m].astype(np.float64)
    return y.astype(np.float32)


@dataclasses.dataclass(frozen=True)
class Config:
    """One entry of BASELINE.json `configs`."""
    name: str
    N: int
    M: int
    K: int
    dictionary: str          # 'gaussian' | 'bernoulli'
    values: str              # see sparse_signal
    eps: float
    max_iter: int
    B: int = 1               # signals sharing the dictionary


def config(name: str) -> Config:
    """cfg1, cfg2, cfg3, cfg5, and cfg4_<M> for M in {2048,...,32768}."""
    if name == "cfg1":
        return Config(name, 256, 1024, 16, "gaussian", "normal", 1e-5, 4096)
    if name == "cfg2":
        return Config(name, 2048, 8192, 128, "gaussian", "pm_uniform", 1e-5, 16384)
    if name == "cfg3":
        return Config(name, 4096, 16384, 256, "bernoulli", "normal", 1e-5, 32768)
    if name.startswith("cfg4_"):
        M = int(name[5:])
        N = M // 4
        K = N // 16
        return Config(name, N, M, K, "gaussian", "normal", 0.0, 4 * K)
    if name == "cfg5":
        return Config(name, 2048, 8192, 128, "gaussian", "normal", 1e-5, 16384, B=64)
    raise KeyError(name)


def make_dictionary(cfg: Config, seed: int) -> np.ndarray:
    """Raw (un-normalised) atom-major dictionary for a config."""
    if cfg.dictionary == "gaussian":
        return gaussian_dictionary(cfg.N, cfg.M, seed)
    if cfg.dictionary == "bernoulli":
        return bernoulli_dictionary(cfg.N, cfg.M, seed)
    raise ValueError(cfg.dictionary)


def make_signals(cfg: Config, psi_t_normalised: np.ndarray, seed: int):
    """X[B, M] float64 (true sparse signals), supports[B, K], Y[B, N] float32, drawn for
    the dictionary bits actually used by the solver (i.e. AFTER column normalisation)."""
    X = np.zeros((cfg.B, cfg.M), dtype=np.float64)
    S = np.zeros((cfg.B, cfg.K), dtype=np.int64)
    Y = np.zeros((cfg.B, cfg.N), dtype=np.float32)
    for b in range(cfg.B):
        X[b], S[b] = sparse_signal(cfg.M, cfg.K, seed, cfg.values, signal=b)
        Y[b] = encode(psi_t_normalised, X[b], S[b])
    return X, S, Y
