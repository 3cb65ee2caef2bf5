"""Seeded synthetic inputs shaped like the paper's workloads.

This package is the ONE piece shared by the CPU oracle's tests and the CUDA path's tests/bench:
it produces the inputs (H in BSR and CSR form, X, permutations) and nothing else.  It contains
none of the method's arithmetic and imports neither ``oracle`` nor ``paper_2110_15853_b200``.

The generators are counter-based (see ``synth.c``): every entry is a pure function of
(seed, stream, i, j), so the same arrays come out on any host and any thread count.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth.c")

STREAM_A, STREAM_MASK, STREAM_DIAG, STREAM_X, STREAM_PERM = 1, 2, 3, 4, 5
STREAM_U = 6       # adjoint-check probe vectors
STREAM_V0 = 7      # Lanczos start vector
STREAM_COLS = 8    # column sample


def build(force: bool = False) -> str:
    """Compile synth.c into synth/_build/libsynth-<hash>.so (portable flags, OpenMP)."""
    with open(_SRC, "rb") as f:
        tag = hashlib.sha1(f.read()).hexdigest()[:12]
    out_dir = os.path.join(_HERE, "_build")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"libsynth-{tag}.so")
    if force or not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, so)
    return so


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
        i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
        f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
        c_i32, c_i64, c_u64, c_f64 = ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double
        L.synth_uniform.restype = c_f64
        L.synth_uniform.argtypes = [c_u64] * 4
        L.synth_normal.restype = c_f64
        L.synth_normal.argtypes = [c_u64] * 4
        L.synth_num_blocks.restype = c_i64
        L.synth_num_blocks.argtypes = [c_i32]
        L.synth_bsr_structure.restype = None
        L.synth_bsr_structure.argtypes = [c_i32, i32p, i32p]
        L.synth_bsr_values.restype = None
        L.synth_bsr_values.argtypes = [c_i32, c_i32, c_f64, c_u64, i32p, i32p, f64p]
        L.synth_bsr_count_nnz.restype = None
        L.synth_bsr_count_nnz.argtypes = [c_i64, c_i32, i32p, i32p, f64p, i64p]
        L.synth_bsr_to_csr_nonzeros.restype = None
        L.synth_bsr_to_csr_nonzeros.argtypes = [c_i64, c_i32, i32p, i32p, f64p, i32p, i32p, f64p]
        L.synth_dense_normal.restype = None
        L.synth_dense_normal.argtypes = [c_i64, c_i64, c_i64, c_i64, c_u64, c_u64, ctypes.c_void_p]
        L.synth_permutation.restype = None
        L.synth_permutation.argtypes = [c_i64, c_u64, i32p]
        L.synth_permute_csr.restype = None
        L.synth_permute_csr.argtypes = [c_i64, i32p, i32p, f64p, i32p, i32p, i32p, f64p]
        L.synth_permute_rows.restype = None
        L.synth_permute_rows.argtypes = [c_i64, c_i64, f64p, c_i64, i32p, f64p, c_i64]
        L.synth_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


@dataclass(frozen=True)
class Config:
    """One of BASELINE.json's synthetic workloads."""
    name: str
    G: int            # subdomains per side
    b: int            # localized basis functions per subdomain (block size)
    z: float          # fraction of off-diagonal-block entries zeroed (L1-localization sparsity)
    N: int            # wavefunction columns
    m: int            # Chebyshev degree
    seed: int
    panel: int = 0    # column-panel width (0 = whole block)

    @property
    def nb(self) -> int:
        return self.G ** 3

    @property
    def M(self) -> int:
        return self.nb * self.b


# BASELINE.json "configs" 1-4 (config 5 reuses config 3's H)
CONFIGS = {
    "tiny": Config("tiny", G=4, b=32, z=0.0, N=32, m=10, seed=1001),
    "al": Config("al", G=8, b=128, z=0.3, N=1024, m=20, seed=1002),
    "si": Config("si", G=12, b=128, z=0.4, N=4096, m=20, seed=1003),
    "largest": Config("largest", G=16, b=96, z=0.4, N=14336, m=20, seed=1004, panel=2048),
}


@dataclass
class BSR:
    M: int
    b: int
    row_ptr: np.ndarray   # int32 [nb+1]
    col_idx: np.ndarray   # int32 [nblocks]
    values: np.ndarray    # float64 [nblocks, b, b] row-major tiles, explicit zeros kept

    @property
    def nblocks(self) -> int:
        return int(self.col_idx.shape[0])


@dataclass
class CSR:
    M: int
    row_ptr: np.ndarray   # int32 [M+1]
    col_idx: np.ndarray   # int32 [nnz], ascending per row
    values: np.ndarray    # float64 [nnz]

    @property
    def nnz(self) -> int:
        return int(self.col_idx.shape[0])


def hamiltonian_bsr(G: int, b: int, z: float, seed: int) -> BSR:
    """Block-sparse symmetric H on a G^3 open-boundary grid, 27-neighbour coupling."""
    L = lib()
    nb = G ** 3
    nblocks = int(L.synth_num_blocks(G))
    row_ptr = np.empty(nb + 1, np.int32)
    col_idx = np.empty(nblocks, np.int32)
    L.synth_bsr_structure(G, row_ptr, col_idx)
    values = np.empty((nblocks, b, b), np.float64)
    L.synth_bsr_values(G, b, float(z), seed, row_ptr, col_idx, values.reshape(-1))
    return BSR(nb * b, b, row_ptr, col_idx, values)


def bsr_to_csr_nonzeros(H: BSR) -> CSR:
    """CSR holding only the non-zero entries of H (what the paper's truncation would store)."""
    L = lib()
    nb = H.M // H.b
    cnt = np.empty(H.M, np.int64)
    flat = H.values.reshape(-1)
    L.synth_bsr_count_nnz(nb, H.b, H.row_ptr, H.col_idx, flat, cnt)
    nnz = int(cnt.sum())
    if nnz >= 2 ** 31:
        raise ValueError("nnz does not fit int32")
    row_ptr = np.zeros(H.M + 1, np.int32)
    np.cumsum(cnt, out=row_ptr[1:])
    col = np.empty(nnz, np.int32)
    val = np.empty(nnz, np.float64)
    L.synth_bsr_to_csr_nonzeros(nb, H.b, H.row_ptr, H.col_idx, flat, row_ptr, col, val)
    return CSR(H.M, row_ptr, col, val)


def dense_normal(M: int, N: int, seed: int, stream: int = STREAM_X, col0: int = 0, out: np.ndarray | None = None) -> np.ndarray:
    """M x N block of N(0,1), entry (i, col0+j) a pure function of (seed, stream, i, col0+j)."""
    if out is None:
        out = np.empty((M, N), np.float64)
    assert out.dtype == np.float64 and out.shape == (M, N) and out.strides[1] == 8
    ld = out.strides[0] // 8 if M > 1 else N
    lib().synth_dense_normal(M, N, ld, col0, seed, stream, out.ctypes.data)
    return out


def permutation(M: int, seed: int) -> np.ndarray:
    p = np.empty(M, np.int32)
    lib().synth_permutation(M, seed, p)
    return p


def permute_csr(H: CSR, perm: np.ndarray) -> CSR:
    """Symmetric permutation H' = P H P^T, H'[perm[i], perm[j]] = H[i, j]."""
    rp = np.empty(H.M + 1, np.int32)
    col = np.empty(H.nnz, np.int32)
    val = np.empty(H.nnz, np.float64)
    lib().synth_permute_csr(H.M, H.row_ptr, H.col_idx, H.values, np.ascontiguousarray(perm, np.int32), rp, col, val)
    return CSR(H.M, rp, col, val)


def permute_rows(X: np.ndarray, perm: np.ndarray) -> np.ndarray:
    """out[perm[i], :] = X[i, :]"""
    X = np.ascontiguousarray(X)
    out = np.empty_like(X)
    lib().synth_permute_rows(X.shape[0], X.shape[1], X, X.shape[1], np.ascontiguousarray(perm, np.int32), out, X.shape[1])
    return out


def split_hybrid(H: CSR, D: int) -> tuple[np.ndarray, CSR]:
    """The paper's two-part layout of the same matrix: (dense diagonal blocks, CSR of the rest).  Block k
    covers rows and columns [k D, min((k + 1) D, M)); the blocks come back as one (ceil(M / D), D, D) array (zeros where H has no
    entry and beyond M).  A layout change only: no arithmetic."""
    M = H.M
    nd = (M + D - 1) // D
    diag = np.zeros((nd, D, D), np.float64)
    rows = np.repeat(np.arange(M, dtype=np.int64), np.diff(H.row_ptr))
    cols = H.col_idx.astype(np.int64)
    inside = (rows // D) == (cols // D)
    diag[rows[inside] // D, rows[inside] % D, cols[inside] % D] = H.values[inside]
    keep = ~inside
    rp = np.zeros(M + 1, np.int64)
    np.add.at(rp, rows[keep] + 1, 1)
    return diag, CSR(M, np.cumsum(rp).astype(np.int32), H.col_idx[keep].copy(), H.values[keep].copy())


def column_sample(N: int, panel: int, count: int, seed: int) -> np.ndarray:
    """Seeded column sample: {0, N-1, every panel's first and last} plus random ones."""
    w = panel if panel > 0 else N
    must = {0, N - 1}
    for c0 in range(0, N, w):
        must.add(c0)
        must.add(min(c0 + w, N) - 1)
    cols = sorted(must)
    L = lib()
    k = 0
    have = set(cols)
    while len(cols) < min(count, N):
        c = int(L.synth_uniform(seed, STREAM_COLS, k, 0) * N)
        k += 1
        if c not in have:
            have.add(c)
            cols.append(c)
    return np.array(sorted(cols[:max(count, len(must))]), np.int64)


def num_threads() -> int:
    return int(lib().synth_num_threads())
