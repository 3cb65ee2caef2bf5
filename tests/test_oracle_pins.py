"""Pins P1-P6 for the CPU oracle: the oracle is checked against things other
than itself -- dense library products, the Chebyshev closed form, a known eigendecomposition,
degenerate matrices, algebraic invariants, and numpy's symmetric eigensolver."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "cheb_scalar_pins.txt")


def relerr(A, B):
    d = np.linalg.norm(A - B)
    n = np.linalg.norm(B)
    return d / n if n > 0 else d


def dense_to_csr(Hd, keep_zeros=False):
    M = Hd.shape[0]
    rp = np.zeros(M + 1, np.int32)
    cols, vals = [], []
    for i in range(M):
        idx = np.arange(M) if keep_zeros else np.nonzero(Hd[i])[0]
        cols.append(idx.astype(np.int32))
        vals.append(Hd[i, idx])
        rp[i + 1] = rp[i] + len(idx)
    return rp, np.concatenate(cols).astype(np.int32) if cols else np.zeros(0, np.int32), \
        np.concatenate(vals).astype(np.float64) if vals else np.zeros(0)


def diag_csr(d):
    M = len(d)
    return np.arange(M + 1, dtype=np.int32), np.arange(M, dtype=np.int32), np.asarray(d, np.float64).copy()


def cheb_T(m, t):
    """Closed form of the Chebyshev polynomial of the first kind."""
    if abs(t) <= 1.0:
        return math.cos(m * math.acos(t))
    s = 1.0 if (t > 0 or m % 2 == 0) else -1.0
    return s * math.cosh(m * math.acosh(abs(t)))


def p_closed(m, lam, a, b, a0):
    e, c = (b - a) / 2, (b + a) / 2
    return cheb_T(m, (lam - c) / e) / cheb_T(m, (a0 - c) / e)


def random_sym_sparse(M, density, rng):
    A = rng.standard_normal((M, M)) * (rng.random((M, M)) < density)
    return (A + A.T) / 2


# ------------------------------------------------------------------ P1: dense brute force
@pytest.mark.parametrize("M,N,density", [(1, 1, 1.0), (7, 3, 0.5), (64, 33, 0.1), (256, 17, 0.05), (50, 5, 0.0)])
def test_p1_spmm_vs_dense(M, N, density):
    rng = np.random.default_rng(M * 1000 + N)
    Hd = random_sym_sparse(M, density, rng)
    if M > 8:
        Hd[3, :] = 0.0
        Hd[:, 3] = 0.0          # an empty row/column
    X = rng.standard_normal((M, N))
    rp, col, val = dense_to_csr(Hd)
    ref = Hd @ X                # library routine, independent of the oracle
    assert relerr(oracle.spmm(rp, col, val, 1.0, X), ref) <= 1e-14
    assert relerr(oracle.dense_hx(Hd, X), ref) <= 1e-14
    Y0 = rng.standard_normal((M, N))
    got = oracle.spmm(rp, col, val, -0.75, X, 2.5, Y0.copy())
    assert relerr(got, -0.75 * ref + 2.5 * Y0) <= 1e-14
    # beta == 0 must not read Y (NaN-safe)
    Yn = np.full((M, N), np.nan)
    got = oracle.spmm(rp, col, val, 1.0, X, 0.0, Yn)
    assert np.isfinite(got).all()


def test_p1_strided_views():
    rng = np.random.default_rng(5)
    M, N = 40, 6
    Hd = random_sym_sparse(M, 0.3, rng)
    rp, col, val = dense_to_csr(Hd)
    Xbig = rng.standard_normal((M, 11))
    X = Xbig[:, 2:2 + N]        # leading dimension 11
    assert relerr(oracle.spmm(rp, col, val, 1.0, X), Hd @ X) <= 1e-14


def test_p1_config1_bsr_and_csr_vs_dense():
    cfg = synth.CONFIGS["tiny"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    X = synth.dense_normal(cfg.M, cfg.N, cfg.seed)
    # dense expansion written here, independently of the oracle's own expansion
    Hd = np.zeros((cfg.M, cfg.M))
    nb = cfg.nb
    for I in range(nb):
        for p in range(H.row_ptr[I], H.row_ptr[I + 1]):
            J = H.col_idx[p]
            Hd[I * cfg.b:(I + 1) * cfg.b, J * cfg.b:(J + 1) * cfg.b] = H.values[p]
    assert np.array_equal(Hd, Hd.T)
    ref = Hd @ X
    rp, col, val = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    assert rp[-1] == H.nblocks * cfg.b * cfg.b            # explicit zeros kept
    assert relerr(oracle.spmm(rp, col, val, 1.0, X), ref) <= 1e-14
    C = synth.bsr_to_csr_nonzeros(H)
    assert relerr(oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, X), ref) <= 1e-14
    assert relerr(oracle.dense_hx(Hd, X), ref) <= 1e-14


def test_p1_bsr_expansion_with_zeros_small():
    rng = np.random.default_rng(11)
    b, nb = 3, 4
    brp = np.array([0, 2, 3, 3, 5], np.int32)        # block row 2 is empty
    bcol = np.array([0, 2, 1, 0, 3], np.int32)
    bval = rng.standard_normal((5, b, b))
    bval[1, 1, :] = 0.0
    Hd = np.zeros((nb * b, nb * b))
    for I in range(nb):
        for p in range(brp[I], brp[I + 1]):
            Hd[I * b:(I + 1) * b, bcol[p] * b:(bcol[p] + 1) * b] = bval[p]
    rp, col, val = oracle.bsr_to_csr(b, brp, bcol, bval)
    X = rng.standard_normal((nb * b, 4))
    assert relerr(oracle.spmm(rp, col, val, 1.0, X), Hd @ X) <= 1e-14
    assert np.all(np.diff(rp)[6:9] == 0)


# ------------------------------------------------------------------ P2: scalar closed form
def read_golden():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            kind, m, arg, expr = line.split()
            val = float(Fraction(expr)) if "/" in expr else float(expr)
            rows.append((kind, int(m), arg, val))
    return rows


def test_p2_golden_scalar_values():
    a0, a, b = 0.0, 2.0, 10.0
    rows = read_golden()
    assert len(rows) >= 20
    # sigma_k of the paper's recurrence, reproduced in exact rational arithmetic
    e, c = Fraction(4), Fraction(6)
    sig = e / (Fraction(0) - c)
    gamma = 2 / sig
    sigmas = {1: sig}
    for k in range(2, 6):
        sig = 1 / (gamma - sig)
        sigmas[k] = sig
    for kind, m, arg, val in rows:
        if kind == "sigma":
            assert float(sigmas[m]) == pytest.approx(val, rel=1e-15)
            # sigma_k = T_{k-1}(t0)/T_k(t0): the scaling that makes p_m(a0) = 1
            assert cheb_T(m - 1, -1.5) / cheb_T(m, -1.5) == pytest.approx(val, rel=1e-13)
    # the oracle on H = diag(lambda): every entry is multiplied by p_m(lambda)
    pts = sorted({float(arg) for kind, _, arg, _ in rows if kind == "p"})
    rp, col, val_ = diag_csr(pts)
    X = np.arange(1, len(pts) * 3 + 1, dtype=np.float64).reshape(len(pts), 3) / 7.0
    for m in sorted({m for kind, m, _, _ in rows if kind == "p"}):
        Y = oracle.cheb_filter(rp, col, val_, X, m, a, b, a0)
        for kind, mm, arg, expected in rows:
            if kind != "p" or mm != m:
                continue
            i = pts.index(float(arg))
            got = Y[i] / X[i]
            if expected == 0.0:
                assert np.all(np.abs(got) <= 1e-15)
            else:
                assert np.allclose(got, expected, rtol=1e-13, atol=0), (m, arg, got, expected)


@pytest.mark.parametrize("m", [1, 2, 3, 5, 10, 11, 20])
def test_p2_diagonal_closed_form(m):
    rng = np.random.default_rng(m)
    a0, a, b = -0.3, 1.7, 20.4
    d = np.concatenate([rng.uniform(a0, b, 60), [a0, a, b, (a + b) / 2, a0 - 0.05]])
    X = rng.standard_normal((len(d), 4))
    rp, col, val = diag_csr(d)
    Y = oracle.cheb_filter(rp, col, val, X, m, a, b, a0)
    P = np.array([p_closed(m, lam, a, b, a0) for lam in d])
    assert relerr(Y, P[:, None] * X) <= 1e-13
    Yl = oracle.cheb_filter(rp, col, val, X, m, a, b, a0, long_double=True)
    assert relerr(Yl, P[:, None] * X) <= 1e-13


# ------------------------------------------------------------------ P3: known eigendecomposition
@pytest.mark.parametrize("M,m,fmt", [(64, 10, "csr"), (128, 20, "bsr"), (256, 7, "csr")])
def test_p3_eigendecomposition(M, m, fmt):
    rng = np.random.default_rng(M + m)
    a0, a, b = 0.0, 3.0, 12.0
    Q, _ = np.linalg.qr(rng.standard_normal((M, M)))
    lam = np.concatenate([rng.uniform(a0, a, M // 4), rng.uniform(a, b, M - M // 4 - 4), [a0, a, b, a0 - 0.01]])
    Hd = (Q * lam) @ Q.T
    Hd = (Hd + Hd.T) / 2
    X = rng.standard_normal((M, 9))
    P = np.array([p_closed(m, l, a, b, a0) for l in lam])
    ref = (Q * P) @ (Q.T @ X)
    if fmt == "csr":
        rp, col, val = dense_to_csr(Hd, keep_zeros=True)
    else:
        bs = 16
        nb = M // bs
        brp = np.arange(0, nb * nb + 1, nb, dtype=np.int32)
        bcol = np.tile(np.arange(nb, dtype=np.int32), nb)
        bval = Hd.reshape(nb, bs, nb, bs).transpose(0, 2, 1, 3).reshape(nb * nb, bs, bs).copy()
        rp, col, val = oracle.bsr_to_csr(bs, brp, bcol, bval)
    Y = oracle.cheb_filter(rp, col, val, X, m, a, b, a0)
    assert relerr(Y, ref) <= 1e-11


# ------------------------------------------------------------------ P4: degenerate matrices
@pytest.mark.parametrize("m", [1, 2, 3, 4, 10, 11])
def test_p4_degenerate(m):
    rng = np.random.default_rng(40 + m)
    M = 12
    a0, a, b = -1.0, 2.0, 9.0
    e, c = (b - a) / 2, (b + a) / 2
    t0 = (a0 - c) / e
    X = rng.standard_normal((M, 3))
    Tm = cheb_T(m, t0)

    def filt(dval):
        rp, col, val = diag_csr(np.full(M, dval))
        return oracle.cheb_filter(rp, col, val, X, m, a, b, a0)

    assert relerr(filt(a0), X) <= 1e-13                               # p_m(a0) = 1
    if m % 2:
        assert np.linalg.norm(filt(c)) <= 1e-13 * np.linalg.norm(X)   # T_m(0) = 0, m odd
    else:
        assert relerr(filt(c), ((-1) ** (m // 2)) * X / Tm) <= 1e-13  # T_m(0) = (-1)^(m/2)
    assert relerr(filt(b), X / Tm) <= 1e-13                           # T_m(1) = 1
    assert relerr(filt(a), X / abs(Tm)) <= 1e-13                      # T_m(-1) = (-1)^m


def test_p4_m0_m1_m2_by_definition():
    rng = np.random.default_rng(3)
    M, N = 48, 5
    Hd = random_sym_sparse(M, 0.2, rng) + np.diag(rng.uniform(0, 10, M))
    rp, col, val = dense_to_csr(Hd)
    X = rng.standard_normal((M, N))
    a0, a, b = -2.0, 3.0, 13.0
    e, c = (b - a) / 2, (b + a) / 2
    assert np.array_equal(oracle.cheb_filter(rp, col, val, X, 0, a, b, a0), X)
    Y1 = oracle.cheb_filter(rp, col, val, X, 1, a, b, a0)
    assert relerr(Y1, (Hd @ X - c * X) / (a0 - c)) <= 1e-13
    S = (Hd - c * np.eye(M)) / e
    t0 = (a0 - c) / e
    Y2 = oracle.cheb_filter(rp, col, val, X, 2, a, b, a0)
    assert relerr(Y2, (2 * S @ (S @ X) - X) / (2 * t0 * t0 - 1)) <= 1e-13
    # single fused step: alpha*(H Yk - c Yk) + beta*Ykm1
    Z = rng.standard_normal((M, N))
    got = oracle.cheb_step(rp, col, val, 0.37, c, -0.21, X, Z)
    assert relerr(got, 0.37 * (Hd @ X - c * X) - 0.21 * Z) <= 1e-14
    got = oracle.cheb_step(rp, col, val, 0.37, c, 123.0, X, None)
    assert relerr(got, 0.37 * (Hd @ X - c * X)) <= 1e-14
    with pytest.raises(ValueError):
        oracle.cheb_filter(rp, col, val, X, -1, a, b, a0)
    with pytest.raises(ValueError):
        oracle.cheb_filter(rp, col, val, X, 3, a, a, a0)
    with pytest.raises(ValueError):
        oracle.cheb_filter(rp, col, val, X, 3, a, b, a + 1)


# ------------------------------------------------------------------ P5: invariants
@pytest.fixture(scope="module")
def tiny():
    cfg = synth.CONFIGS["tiny"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    C = synth.bsr_to_csr_nonzeros(H)
    v0 = synth.dense_normal(cfg.M, 1, cfg.seed, synth.STREAM_V0).reshape(-1)
    a, b, a0 = oracle.filter_bounds(C.row_ptr, C.col_idx, C.values, v0, cfg.N)
    return cfg, H, C, (a, b, a0)


def test_p5_invariants(tiny):
    cfg, H, C, (a, b, a0) = tiny
    m = cfg.m
    F = lambda X: oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, b, a0)
    U = synth.dense_normal(cfg.M, 6, 77, synth.STREAM_U)
    V = synth.dense_normal(cfg.M, 6, 78, synth.STREAM_U)
    FU, FV = F(U), F(V)
    # linearity
    assert relerr(F(1.5 * U - 0.25 * V), 1.5 * FU - 0.25 * FV) <= 1e-12
    # self-adjointness: U^T F(V) = (V^T F(U))^T  (F is a polynomial in symmetric H)
    A, B = U.T @ FV, (V.T @ FU).T
    assert np.linalg.norm(A - B) <= 1e-12 * np.linalg.norm(U) * np.linalg.norm(FV)
    # column independence: a column subset reproduces those columns bit for bit
    sub = F(np.ascontiguousarray(U[:, [1, 4]]))
    assert np.array_equal(sub, FU[:, [1, 4]])
    # permutation equivariance F_{PHP^T}(PX) = P F_H(X)
    perm = synth.permutation(cfg.M, 9)
    Cp = synth.permute_csr(C, perm)
    Yp = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, synth.permute_rows(U, perm), m, a, b, a0)
    assert relerr(Yp, synth.permute_rows(FU, perm)) <= 1e-12
    # BSR (explicit zeros) and CSR (non-zeros only) inputs give the same filter
    rp, col, val = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    assert relerr(oracle.cheb_filter(rp, col, val, U, m, a, b, a0), FU) <= 1e-13
    # long-double error budget
    FUl = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, U, m, a, b, a0, long_double=True)
    assert relerr(FU, FUl) <= 1e-13


def test_p5_boundedness(tiny):
    """|p_k| <= 1 on [a0, b] (the overflow guard of PAPER.md:L232): no column norm may grow."""
    cfg, H, C, (a, b, a0) = tiny
    X = synth.dense_normal(cfg.M, 8, cfg.seed)
    n0 = np.linalg.norm(X, axis=0)
    for m in (1, 2, 5, 10):
        Y = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, b, a0)
        assert np.all(np.linalg.norm(Y, axis=0) <= n0 * (1 + 1e-12))


def test_p5_damping_of_unwanted_components(tiny):
    """Eigen-components in [a, b] shrink by >= |T_m(t0)| relative to the a0 end."""
    cfg, H, C, (a, b, a0) = tiny
    Hd = np.zeros((cfg.M, cfg.M))
    for i in range(cfg.M):
        Hd[i, C.col_idx[C.row_ptr[i]:C.row_ptr[i + 1]]] = C.values[C.row_ptr[i]:C.row_ptr[i + 1]]
    w, Q = np.linalg.eigh(Hd)
    assert a0 <= w[0] and w[-1] <= b
    X = synth.dense_normal(cfg.M, 4, 5)
    m = cfg.m
    Y = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, b, a0)
    P = np.array([p_closed(m, l, a, b, a0) for l in w])
    assert relerr(Y, (Q * P) @ (Q.T @ X)) <= 1e-11
    Tm = abs(cheb_T(m, (a0 - (a + b) / 2) / ((b - a) / 2)))
    coef = Q.T @ Y
    coef0 = Q.T @ X
    unwanted = w >= a
    assert np.all(np.abs(coef[unwanted]) <= np.abs(coef0[unwanted]) / Tm * (1 + 1e-9) + 1e-14)


# ------------------------------------------------------------------ P6: Lanczos bounds
def test_p6_lanczos_bounds_config1(tiny):
    cfg, H, C, (a, b, a0) = tiny
    Hd = np.zeros((cfg.M, cfg.M))
    for i in range(cfg.M):
        Hd[i, C.col_idx[C.row_ptr[i]:C.row_ptr[i + 1]]] = C.values[C.row_ptr[i]:C.row_ptr[i + 1]]
    w = np.linalg.eigvalsh(Hd)
    assert a0 <= w[0] and b >= w[-1]
    assert a0 > w[0] - 1.0 and b < w[-1] + 1.0          # and not uselessly loose
    assert a0 < a < b
    assert np.sum(w < a) >= cfg.N // 4                  # wanted states do fall below a
    v0 = synth.dense_normal(cfg.M, 1, cfg.seed, synth.STREAM_V0).reshape(-1)
    _, _, info = oracle.lanczos_bounds(C.row_ptr, C.col_idx, C.values, v0, 30)
    k = len(info["alpha"])
    T = np.diag(info["alpha"]) + np.diag(info["beta"][:k - 1], 1) + np.diag(info["beta"][:k - 1], -1)
    th, Z = np.linalg.eigh(T)
    assert np.allclose(info["theta"], th, rtol=0, atol=1e-12 * max(1.0, abs(th).max()))
    assert np.allclose(np.abs(info["zlast"]), np.abs(Z[-1, :]), atol=1e-10)


def test_p6_lanczos_small_dense():
    rng = np.random.default_rng(8)
    M = 96
    Hd = random_sym_sparse(M, 0.3, rng) + np.diag(rng.uniform(0, 20, M))
    rp, col, val = dense_to_csr(Hd)
    w = np.linalg.eigvalsh(Hd)
    a0, b, info = oracle.lanczos_bounds(rp, col, val, rng.standard_normal(M), 30)
    assert a0 <= w[0] + 1e-12 and b >= w[-1] - 1e-12
    # first Lanczos coefficient is the Rayleigh quotient of v0
    v0 = rng.standard_normal(M)
    _, _, info = oracle.lanczos_bounds(rp, col, val, v0, 5)
    assert info["alpha"][0] == pytest.approx(v0 @ Hd @ v0 / (v0 @ v0), rel=1e-13)


# ------------------------------------------------------------------ P7: subspace projection (NEXT-1)
# oracle.gram / oracle.project pinned by hand-computed integers, numpy's matmul,
# a known eigendecomposition and three identities a transposed operand or a dropped term would break.
def read_gram_golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "gram_pins.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if not line:
                continue
            r, c = int(line[1]), int(line[2])
            out[line[0]] = np.array([float(v) for v in line[3:]], np.float64).reshape(r, c)
    return out


def test_p7_hand_computed_projection():
    g = read_gram_golden()
    assert np.array_equal(oracle.gram(g["X"], g["W"]), g["XtW"])          # not symmetric: catches a transposed operand
    rp, col, val = dense_to_csr(g["H"], keep_zeros=False)
    assert np.array_equal(oracle.spmm(rp, col, val, 1.0, g["X"]), g["HX"])
    assert np.array_equal(oracle.project(rp, col, val, g["X"]), g["XtHX"])


@pytest.mark.parametrize("M,n", [(1, 1), (5, 3), (257, 33), (1000, 64), (0, 4)])
def test_p7_gram_vs_numpy(M, n):
    rng = np.random.default_rng(100 * M + n)
    X, W = rng.standard_normal((M, n)), rng.standard_normal((M, n))
    G = oracle.gram(X, W)
    ref = X.T @ W
    assert np.linalg.norm(G - ref) <= 1e-14 * max(1.0, np.linalg.norm(ref))
    # strided views (leading dimension > n)
    Xp, Wp = np.zeros((M, n + 3)), np.zeros((M, n + 5))
    Xp[:, :n], Wp[:, :n] = X, W
    assert np.array_equal(oracle.gram(Xp[:, :n], Wp[:, :n]), G)


def test_p7_projection_of_eigenvectors_is_diagonal():
    """H = Q Lambda Q^T, X = n columns of Q  =>  X^T H X = diag(lambda) exactly (up to rounding)."""
    rng = np.random.default_rng(7)
    M, n = 128, 17
    Q, _ = np.linalg.qr(rng.standard_normal((M, M)))
    lam = rng.uniform(-1.0, 20.0, M)
    Hd = (Q * lam) @ Q.T
    Hd = (Hd + Hd.T) / 2
    rp, col, val = dense_to_csr(Hd, keep_zeros=True)
    cols = rng.permutation(M)[:n]
    G = oracle.project(rp, col, val, np.ascontiguousarray(Q[:, cols]))
    assert np.linalg.norm(G - np.diag(lam[cols])) <= 1e-12 * np.linalg.norm(lam)


def test_p7_projection_identities(tiny):
    _cfg, H, C, _bounds = tiny
    rng = np.random.default_rng(11)
    n = 12
    X = rng.standard_normal((H.M, n))
    G = oracle.project(C.row_ptr, C.col_idx, C.values, X)
    nG = np.linalg.norm(G)
    assert np.linalg.norm(G - G.T) <= 1e-13 * nG                          # H symmetric => H_F symmetric
    R = rng.standard_normal((n, n))
    G2 = oracle.project(C.row_ptr, C.col_idx, C.values, X @ R)           # congruence: (XR)^T H (XR) = R^T G R
    assert np.linalg.norm(G2 - R.T @ G @ R) <= 1e-12 * np.linalg.norm(G2)
    # trace identity: tr(X^T H X) = sum_e h_e * <X[row_e,:], X[col_e,:]>
    rows = np.repeat(np.arange(H.M), np.diff(C.row_ptr))
    tr = float(np.sum(C.values * np.einsum("ij,ij->i", X[rows], X[C.col_idx])))
    assert abs(np.trace(G) - tr) <= 1e-12 * abs(tr)


# ------------------------------------------------------------------ P8: rotation Y = X Q (Algorithm 1 step 5)
def test_p8_rotate_pins():
    g = read_gram_golden()
    assert np.array_equal(oracle.rotate(g["X"], g["Qrot"]), g["XQ"])       # hand-computed, non-square Q
    rng = np.random.default_rng(8)
    for M, K, n in [(1, 1, 1), (7, 5, 3), (300, 130, 70), (64, 257, 33)]:
        X, Q = rng.standard_normal((M, K)), rng.standard_normal((K, n))
        Y = oracle.rotate(X, Q)
        ref = X @ Q
        assert np.linalg.norm(Y - ref) <= 1e-14 * max(1.0, np.linalg.norm(ref))
    X = rng.standard_normal((50, 9))
    assert np.array_equal(oracle.rotate(X, np.eye(9)), X)                 # Q = I
    perm = rng.permutation(9)
    assert np.array_equal(oracle.rotate(X, np.ascontiguousarray(np.eye(9)[:, perm])), X[:, perm])   # a column permutation is exact
    Q = rng.standard_normal((9, 9))
    G = oracle.gram(X, X)
    Y = oracle.rotate(X, Q)
    lhs = oracle.gram(Y, Y)                                               # (XQ)^T (XQ) = Q^T (X^T X) Q
    assert np.linalg.norm(lhs - Q.T @ G @ Q) <= 1e-12 * np.linalg.norm(lhs)


# ------------------------------------------------------------------ P9: orthonormalisation X_F = Orth(X) (Algorithm 1 step 2)
def test_p9_gram_schmidt_pins():
    g = read_gram_golden()
    assert np.linalg.norm(oracle.orthonormalize(g["Xgs"]) - g["Qgs"]) <= 1e-15          # hand-computed
    rng = np.random.default_rng(9)
    for M, n, cond in [(5, 3, 1.0), (200, 17, 1.0), (300, 40, 1e6)]:
        X = rng.standard_normal((M, n))
        if cond > 1.0:                                            # ill-conditioned: graded singular values
            U, _, Vt = np.linalg.svd(X, full_matrices=False)
            X = (U * np.logspace(0, -np.log10(cond), n)) @ Vt
        Q = oracle.orthonormalize(X)
        Qn, Rn = np.linalg.qr(X)                                  # library QR, signs fixed so that diag(R) > 0
        sgn = np.sign(np.diag(Rn))
        assert np.linalg.norm(Q - Qn * sgn) <= 1e-13 * cond * np.sqrt(n)
        assert np.linalg.norm(Q.T @ Q - np.eye(n)) <= 1e-14 * n   # orthonormal to rounding level, whatever cond(X)
        R = Q.T @ X
        assert np.linalg.norm(np.tril(R, -1)) <= 1e-13 * np.linalg.norm(R) and np.all(np.diag(R) > 0)
        assert np.linalg.norm(Q @ R - X) <= 1e-13 * np.linalg.norm(X)
    with pytest.raises(np.linalg.LinAlgError):
        oracle.orthonormalize(np.zeros((4, 2)))


# ------------------------------------------------------------------ P10: subdomain recovery for unlabelled, permuted CSR (A0; reading #18)
def _canonical(labels):
    """Partition written canonically: every row gets the smallest row index of its group."""
    labels = np.asarray(labels)
    first = {}
    for i, l in enumerate(labels):
        first.setdefault(int(l), i)
    return np.array([first[int(l)] for l in labels])


def _planted(G, b, z, seed):
    from oracle.recover import recover_subdomains  # noqa: F401
    H = synth.hamiltonian_bsr(G, b, z, seed)
    C = synth.bsr_to_csr_nonzeros(H)
    perm = synth.permutation(H.M, seed + 50)
    Cp = synth.permute_csr(C, perm)
    truth = np.empty(H.M, np.int32)
    truth[perm] = (np.arange(H.M) // b).astype(np.int32)
    return H, C, Cp, truth


@pytest.mark.parametrize("G,b,z", [(3, 8, 0.0), (3, 32, 0.0), (3, 16, 0.4), (3, 32, 0.4), (4, 8, 0.3)])
def test_p10_recover_planted_partition(G, b, z):
    from oracle.recover import recover_subdomains
    H, C, Cp, truth = _planted(G, b, z, 7100 + b)
    labels, n = recover_subdomains(Cp.row_ptr, Cp.col_idx)
    assert n == G ** 3
    assert np.array_equal(_canonical(labels), _canonical(truth))          # the planted partition, exactly
    assert np.array_equal(np.bincount(labels), np.full(n, b))
    # labels are numbered by the smallest row index of the group
    firsts = [int(np.flatnonzero(labels == k)[0]) for k in range(n)]
    assert firsts == sorted(firsts)
    # unpermuted input: the groups are the generator's blocks, numbered in order
    labels0, n0 = recover_subdomains(C.row_ptr, C.col_idx)
    assert n0 == G ** 3 and np.array_equal(labels0, np.arange(H.M) // b)


def test_p10_recover_closed_forms_and_invariants():
    from oracle.recover import recover_subdomains
    # z = 0: rows of a subdomain have identical column sets, so the groups are the classes of equal rows (closed form)
    H, C, Cp, truth = _planted(3, 8, 0.0, 7200)
    rows = [tuple(Cp.col_idx[Cp.row_ptr[i]:Cp.row_ptr[i + 1]]) for i in range(Cp.M)]
    classes = {}
    for i, r in enumerate(rows):
        classes.setdefault(r, i)
    labels, n = recover_subdomains(Cp.row_ptr, Cp.col_idx)
    assert np.array_equal(_canonical(labels), np.array([classes[r] for r in rows]))
    # the library step (A A^T) and plain set intersections give the same labels
    labels_sets, n_sets = recover_subdomains(Cp.row_ptr, Cp.col_idx, counts="sets")
    assert n_sets == n and np.array_equal(labels_sets, labels)
    # a diagonal matrix: M singletons, label(i) = i
    M = 37
    labels, n = recover_subdomains(np.arange(M + 1, dtype=np.int32), np.arange(M, dtype=np.int32))
    assert n == M and np.array_equal(labels, np.arange(M))
    # an empty row and a row without a diagonal entry are singletons / still grouped by pattern
    rp = np.array([0, 0, 2, 4, 5], np.int32)
    ci = np.array([2, 3, 1, 3, 3], np.int32)     # rows 1 and 2 point at each other and at 3; row 3 only at itself
    labels, n = recover_subdomains(rp, ci)
    assert labels is not None and labels[0] == 0 and n >= 2
    # two complete cliques of different size joined by nothing: two groups
    k1, k2 = 5, 9
    rp = [0]
    ci = []
    for i in range(k1 + k2):
        grp = range(0, k1) if i < k1 else range(k1, k1 + k2)
        ci += list(grp)
        rp.append(len(ci))
    labels, n = recover_subdomains(np.array(rp, np.int32), np.array(ci, np.int32))
    assert n == 2 and np.array_equal(labels, np.array([0] * k1 + [1] * k2))
    # G = 2, z = 0: every subdomain neighbours every other, H is fully dense and all rows look alike: "no structure"
    H, C, Cp, truth = _planted(2, 32, 0.0, 7300)
    assert recover_subdomains(Cp.row_ptr, Cp.col_idx) == (None, 0)
    # a candidate set above the cap (one dense 200-clique): reported as "no structure"
    k = 200
    rp = np.arange(0, k * k + 1, k, dtype=np.int32)
    ci = np.tile(np.arange(k, dtype=np.int32), k)
    labels, n = recover_subdomains(rp, ci)
    assert labels is None and n == 0
