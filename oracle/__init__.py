"""CPU oracle for the ChFSI Chebyshev filter -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2110_15853_b200``) never does, and this package never imports the product.

The arithmetic lives in ``ttdft_oracle.cpp`` (plain C++17, fp64, ``-ffp-contract=off``), written
from PAPER.md Algorithm 1 step 1 (L214-223).  This file only compiles it (per host CPU, because
of ``-march=native``) and marshals numpy arrays.  Pins: tests/test_oracle_pins.py (P1-P6);
nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import platform
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ttdft_oracle.cpp")
CXXFLAGS = ["-O3", "-march=native", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-fPIC", "-shared"]


def _host_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        src = f.read()
    return hashlib.sha1(src + flags.encode() + platform.machine().encode() + " ".join(CXXFLAGS).encode()).hexdigest()[:12]


def build(force: bool = False) -> str:
    out_dir = os.path.join(_HERE, "_build")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"liboracle-{_host_tag()}.so")
    if force or not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *CXXFLAGS, "-o", tmp, _SRC])
        os.replace(tmp, so)
    return so


_lib = None
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i64, i32, f64, vp = ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_void_p
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_dense_hx.restype = None
        L.oracle_dense_hx.argtypes = [i64, _f64p, vp, i64, vp, i64, i64]
        L.oracle_bsr_to_csr.restype = None
        L.oracle_bsr_to_csr.argtypes = [i64, i32, _i32p, _i32p, _f64p, _i32p, _i32p, _f64p]
        L.oracle_spmm_csr.restype = None
        L.oracle_spmm_csr.argtypes = [i64, _i32p, _i32p, _f64p, f64, vp, i64, f64, vp, i64, i64]
        L.oracle_cheb_step_csr.restype = None
        L.oracle_cheb_step_csr.argtypes = [i64, _i32p, _i32p, _f64p, f64, f64, f64, vp, i64, vp, i64, vp, i64, i64]
        for name in ("oracle_cheb_filter_csr", "oracle_cheb_filter_csr_ld"):
            fn = getattr(L, name)
            fn.restype = ctypes.c_int
            fn.argtypes = [i64, _i32p, _i32p, _f64p, vp, i64, vp, i64, i64, i32, f64, f64, f64]
        L.oracle_lanczos_bounds.restype = ctypes.c_int
        L.oracle_gram.argtypes = [i64, i64, vp, i64, vp, i64, vp, i64]
        L.oracle_rotate.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64]
        L.oracle_rotate.restype = None
        L.oracle_orth_gs.argtypes = [i64, i64, vp, i64, vp, i64, i32]
        L.oracle_orth_gs.restype = ctypes.c_int
        L.oracle_gram.restype = None
        L.oracle_lanczos_bounds.argtypes = [i64, _i32p, _i32p, _f64p, i32, _f64p, _f64p, _f64p, _f64p, _f64p,
                                            ctypes.POINTER(f64), ctypes.POINTER(f64)]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _mat(X: np.ndarray):
    """(pointer, leading dimension) of a row-major float64 matrix view with unit column stride."""
    assert X.dtype == np.float64 and X.ndim == 2 and (X.shape[1] == 1 or X.strides[1] == 8)
    ld = X.strides[0] // 8 if X.shape[0] > 1 else X.shape[1]
    assert ld >= X.shape[1]
    return X.ctypes.data, ld


def dense_hx(Hd: np.ndarray, X: np.ndarray) -> np.ndarray:
    """Brute-force dense product (pin P1)."""
    Hd = np.ascontiguousarray(Hd, np.float64)
    M = Hd.shape[0]
    Y = np.empty((M, X.shape[1]), np.float64)
    xp, ldx = _mat(X)
    yp, ldy = _mat(Y)
    lib().oracle_dense_hx(M, Hd.reshape(-1), xp, ldx, yp, ldy, X.shape[1])
    return Y


def bsr_to_csr(b: int, brow_ptr: np.ndarray, bcol: np.ndarray, bval: np.ndarray):
    """Expand BSR (b x b row-major tiles) to CSR keeping the explicit zeros."""
    nb = brow_ptr.shape[0] - 1
    nblocks = bcol.shape[0]
    rp = np.empty(nb * b + 1, np.int32)
    col = np.empty(nblocks * b * b, np.int32)
    val = np.empty(nblocks * b * b, np.float64)
    lib().oracle_bsr_to_csr(nb, b, np.ascontiguousarray(brow_ptr, np.int32), np.ascontiguousarray(bcol, np.int32),
                            np.ascontiguousarray(bval, np.float64).reshape(-1), rp, col, val)
    return rp, col, val


def spmm(row_ptr, col, val, alpha: float, X: np.ndarray, beta: float = 0.0, Y: np.ndarray | None = None) -> np.ndarray:
    """Y = alpha*H*X + beta*Y from CSR (beta == 0 does not read Y)."""
    M = row_ptr.shape[0] - 1
    if Y is None:
        assert beta == 0.0
        Y = np.empty((M, X.shape[1]), np.float64)
    xp, ldx = _mat(X)
    yp, ldy = _mat(Y)
    lib().oracle_spmm_csr(M, row_ptr, col, val, alpha, xp, ldx, beta, yp, ldy, X.shape[1])
    return Y


def cheb_step(row_ptr, col, val, alpha: float, c: float, beta: float, Yk: np.ndarray, Ykm1: np.ndarray | None) -> np.ndarray:
    """Yout = alpha*(H*Yk - c*Yk) + beta*Ykm1 (Ykm1 None: beta term absent). PAPER.md:L218, L221."""
    M = row_ptr.shape[0] - 1
    out = np.empty((M, Yk.shape[1]), np.float64)
    kp, ldk = _mat(Yk)
    mp, ldm = (None, 0) if Ykm1 is None else _mat(Ykm1)
    op, ldo = _mat(out)
    lib().oracle_cheb_step_csr(M, row_ptr, col, val, alpha, c, beta, kp, ldk, mp, ldm, op, ldo, Yk.shape[1])
    return out


def cheb_filter(row_ptr, col, val, X: np.ndarray, m: int, a: float, b: float, a0: float, long_double: bool = False) -> np.ndarray:
    """Algorithm 1 step 1: degree-m scaled Chebyshev filter of X."""
    M = row_ptr.shape[0] - 1
    Y = np.empty((M, X.shape[1]), np.float64)
    xp, ldx = _mat(X)
    yp, ldy = _mat(Y)
    fn = lib().oracle_cheb_filter_csr_ld if long_double else lib().oracle_cheb_filter_csr
    rc = fn(M, row_ptr, col, val, xp, ldx, yp, ldy, X.shape[1], m, a, b, a0)
    if rc != 0:
        raise ValueError("oracle_cheb_filter: invalid arguments (need m >= 0 and a0 < a < b)")
    return Y


def lanczos_bounds(row_ptr, col, val, v0: np.ndarray, k: int = 30):
    """Residual-corrected Ritz bounds (a0, b) and the Lanczos data (reading #5)."""
    M = row_ptr.shape[0] - 1
    k = min(k, M)
    alpha = np.zeros(k)
    beta = np.zeros(k)
    theta = np.zeros(k)
    zlast = np.zeros(k)
    a0 = ctypes.c_double()
    b = ctypes.c_double()
    kk = lib().oracle_lanczos_bounds(M, row_ptr, col, val, k, np.ascontiguousarray(v0, np.float64), alpha, beta, theta,
                                     zlast, ctypes.byref(a0), ctypes.byref(b))
    if kk < 1:
        raise ValueError("lanczos failed")
    return a0.value, b.value, dict(alpha=alpha[:kk], beta=beta[:kk], theta=theta[:kk], zlast=zlast[:kk])


def filter_bounds(row_ptr, col, val, v0: np.ndarray, ncols: int, k: int = 30):
    """(a, b, a0) for a block of ncols wanted states: a = a0 + (ncols/M)*(b - a0) (reading #5)."""
    M = row_ptr.shape[0] - 1
    a0, b, _ = lanczos_bounds(row_ptr, col, val, v0, k)
    a = a0 + (ncols / M) * (b - a0)
    return a, b, a0


def gram(X: np.ndarray, W: np.ndarray) -> np.ndarray:
    """G = X^T W by the plain definition (oracle_gram)."""
    assert X.shape == W.shape
    M, n = X.shape
    G = np.empty((n, n), np.float64)
    if M == 0:
        G[:] = 0.0
        return G
    xp, ldx = _mat(X)
    wp, ldw = _mat(W)
    gp, ldg = _mat(G)
    lib().oracle_gram(M, n, xp, ldx, wp, ldw, gp, ldg)
    return G


def project(row_ptr, col, val, X: np.ndarray) -> np.ndarray:
    """H_F = X^T (H X) (Algorithm 1 step 3): the oracle's SpMM followed by the oracle's Gram product."""
    return gram(X, spmm(row_ptr, col, val, 1.0, X))


def rotate(X: np.ndarray, Q: np.ndarray) -> np.ndarray:
    """Y = X Q by the plain definition (oracle_rotate; Algorithm 1 step 5)."""
    M, K = X.shape
    assert Q.shape[0] == K
    n = Q.shape[1]
    Y = np.zeros((M, n), np.float64)
    if M == 0:
        return Y
    xp, ldx = _mat(X)
    qp, ldq = _mat(Q)
    yp, ldy = _mat(Y)
    lib().oracle_rotate(M, K, n, xp, ldx, qp, ldq, yp, ldy)
    return Y


def orthonormalize(X: np.ndarray, sweeps: int = 2) -> np.ndarray:
    """X_F = Orth(X) by Gram-Schmidt (oracle_orth_gs; Algorithm 1 step 2)."""
    M, n = X.shape
    Q = np.zeros((M, n), np.float64)
    xp, ldx = _mat(X)
    qp, ldq = _mat(Q)
    rc = lib().oracle_orth_gs(M, n, xp, ldx, qp, ldq, sweeps)
    if rc:
        raise np.linalg.LinAlgError(f"column {rc - 1} is linearly dependent on the previous ones")
    return Q
