"""Shared helpers for the parity tests (inputs from synth, expected values from oracle)."""
from __future__ import annotations

import functools

import numpy as np

import oracle
import synth


def relerr(got: np.ndarray, ref: np.ndarray) -> float:
    n = np.linalg.norm(ref)
    d = np.linalg.norm(got - ref)
    return float(d / n) if n > 0 else float(d)


def worst_col_relerr(got: np.ndarray, ref: np.ndarray) -> float:
    n = np.linalg.norm(ref, axis=0)
    d = np.linalg.norm(got - ref, axis=0)
    n = np.where(n > 0, n, 1.0)
    return float((d / n).max())


@functools.lru_cache(maxsize=4)
def small_problem(G: int, b: int, z: float, seed: int):
    """BSR H, its two CSR forms (explicit zeros kept / non-zeros only) and Lanczos bounds."""
    H = synth.hamiltonian_bsr(G, b, z, seed)
    C = synth.bsr_to_csr_nonzeros(H)
    full = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    v0 = synth.dense_normal(H.M, 1, seed, synth.STREAM_V0).reshape(-1)
    a0, bb, _ = oracle.lanczos_bounds(C.row_ptr, C.col_idx, C.values, v0, 30)
    return H, C, full, (a0, bb)


def bounds_for(a0: float, b: float, N: int, M: int, wide: bool = False):
    a = a0 + (0.25 if wide else N / M) * (b - a0)
    return a, b, a0
