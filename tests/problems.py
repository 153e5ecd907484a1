"""Problem construction shared by the GPU parity tests, smoke() and bench.py (test/harness code).

Everything here is host-side numpy: seeded inputs from paper_0809_1833_b200.synth, columns normalised by
the ORACLE's float64 routine and rounded to fp32 once, so the dictionary bits fed to both sides never
come from the CUDA path.  (The CUDA normalisation kernel is tested separately against the same bits.)
"""
from __future__ import annotations

import dataclasses

import numpy as np

import oracle
from paper_0809_1833_b200 import synth


@dataclasses.dataclass
class Problem:
    cfg: synth.Config
    psi_raw: np.ndarray      # [M, N] float32, as drawn (un-normalised for Gaussian)
    psi32: np.ndarray        # [M, N] float32, column-normalised (Eq. 4) -- what the solver is given
    X: np.ndarray            # [B, M] float64 true signals
    S: np.ndarray            # [B, K] supports
    Y: np.ndarray            # [B, N] float32 measurements y = Psi x


def normalise_on_host(psi_raw: np.ndarray) -> np.ndarray:
    """Eq. 4 in float64 (oracle), rounded to fp32 once."""
    out = np.empty_like(psi_raw, dtype=np.float32)
    rows = max(1, (64 << 20) // (8 * psi_raw.shape[1]))
    for m0 in range(0, psi_raw.shape[0], rows):
        p64, _ = oracle.normalize_columns(psi_raw[m0:m0 + rows])
        out[m0:m0 + rows] = p64.astype(np.float32)
    return out


def make_problem(cfg: synth.Config, seed: int) -> Problem:
    psi_raw = synth.make_dictionary(cfg, seed)
    psi32 = normalise_on_host(psi_raw) if cfg.dictionary == "gaussian" else psi_raw
    X, S, Y = synth.make_signals(cfg, psi32, seed)
    return Problem(cfg, psi_raw, psi32, X, S, Y)


def custom_config(N, M, K, dictionary="gaussian", values="normal", eps=1e-5, max_iter=None, B=1, name="custom"):
    return synth.Config(name, N, M, K, dictionary, values, eps, max_iter if max_iter is not None else 8 * K, B)
