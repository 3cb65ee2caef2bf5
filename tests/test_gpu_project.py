"""GPU parity of the subspace projection (Algorithm 1 step 3, Sec. 4.3):
ttdft_gram (G = X^T W, kernel K4 on the int8 tensor cores) and ttdft_project (G = X^T (H X)) against the CPU oracle.

Tolerance: the projection has no figure in north_star; K4 evaluates every entry exactly from operands rounded to 55
bits below their column maximum, so its error is bounded like an fp64 dot product's (K4) -- the tests hold it
to the per-product tolerance of the SpMM, 1e-12 relative Frobenius, and pin the expected level (<= 1e-14)."""
import os

import numpy as np
import pytest

import oracle
import synth
from util import relerr, small_problem

pytestmark = pytest.mark.gpu

TOL = 1e-12
ACC = 1e-14      # what 55-bit operands with exact accumulation must deliver on these inputs


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2110_15853_b200 as t
    assert torch.cuda.is_available()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("cluster", ["1", "2"])
@pytest.mark.parametrize("M,N,ld", [(2048, 32, 32), (2048, 33, 40), (1000, 70, 70), (300, 1, 2), (4113, 130, 130), (77, 257, 300),
                                    (128 * 300 + 5, 64, 64)])
def test_gram_vs_oracle(tt, M, N, ld, cluster):
    import torch
    os.environ["TTDFT_K4_CLUSTER"] = cluster
    try:
        X = synth.dense_normal(M, N, 301)
        W = synth.dense_normal(M, N, 302) * 3.0 + 0.5
        ref = oracle.gram(X, W)
        Xd = torch.zeros(M, ld, dtype=torch.float64, device="cuda")
        Wd = torch.zeros(M, ld + 2, dtype=torch.float64, device="cuda")
        Xd[:, :N], Wd[:, :N] = dev(X), dev(W)
        Gd = torch.full((N, ld), float("nan"), dtype=torch.float64, device="cuda")
        tt.gram(Xd[:, :N], Wd[:, :N], Gd[:, :N])
        got = Gd[:, :N].cpu().numpy()
        assert relerr(got, ref) <= ACC
        if ld > N:
            assert torch.isnan(Gd[:, N:]).all()              # nothing written outside the view
        # deterministic: chunks are summed in a fixed order, no floating-point atomics
        G2 = torch.empty(N, N, dtype=torch.float64, device="cuda")
        tt.gram(Xd[:, :N], Wd[:, :N], G2)
        assert np.array_equal(G2.cpu().numpy(), got)
    finally:
        os.environ.pop("TTDFT_K4_CLUSTER", None)


def test_gram_same_operand_and_empty(tt):
    import torch
    X = synth.dense_normal(1500, 96, 311)
    G = torch.empty(96, 96, dtype=torch.float64, device="cuda")
    Xd = dev(X)
    tt.gram(Xd, Xd, G)                                       # X^T X (the overlap matrix of the orthonormalisation)
    got = G.cpu().numpy()
    assert relerr(got, oracle.gram(X, X)) <= ACC
    assert np.array_equal(got, got.T)                        # exact integer sums: bit-for-bit symmetric
    E = torch.empty(0, 5, dtype=torch.float64, device="cuda")
    G5 = torch.full((5, 5), 7.0, dtype=torch.float64, device="cuda")
    tt.gram(E, E, G5)
    assert (G5 == 0).all()


def test_gram_column_dynamic_range(tt):
    """Per-column scaling of both operands: columns 40 orders of magnitude apart, a zero column."""
    import torch
    M, N = 3000, 70
    X = synth.dense_normal(M, N, 321) * 10.0 ** np.linspace(-20, 20, N)[None, :]
    W = synth.dense_normal(M, N, 322) * 10.0 ** np.linspace(15, -15, N)[None, :]
    X[:, 4] = 0.0
    ref = oracle.gram(X, W)
    G = torch.empty(N, N, dtype=torch.float64, device="cuda")
    tt.gram(dev(X), dev(W), G)
    got = G.cpu().numpy()
    assert np.all(got[4, :] == 0.0)
    # entry-wise against the scale of each entry: |x_j| |w_l|
    scale = np.outer(np.linalg.norm(X, axis=0), np.linalg.norm(W, axis=0))
    scale[scale == 0] = 1.0
    assert np.max(np.abs(got - ref) / scale) <= 1e-15 * np.sqrt(M)


@pytest.mark.parametrize("G_,b,z,N", [(4, 32, 0.0, 32), (3, 64, 0.3, 200), (2, 96, 0.4, 130), (3, 128, 0.4, 300)])
def test_project_vs_oracle(tt, G_, b, z, N):
    import torch
    H, C, _, _ = small_problem(G_, b, z, 2000 + b if b != 32 else 1001)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    X = synth.dense_normal(H.M, N, 331)
    ref = oracle.project(C.row_ptr, C.col_idx, C.values, X)
    Gd = torch.empty(N, N, dtype=torch.float64, device="cuda")
    n0 = tt.launch_count()
    tt.project(Hd, dev(X), Gd)
    assert tt.launch_count() - n0 >= 6                       # step + 2 colmax + 2 digit passes + gram + reduce
    got = Gd.cpu().numpy()
    assert relerr(got, ref) <= TOL
    assert relerr(got, got.T) <= 1e-13                       # symmetric up to rounding (H is symmetric)
    # the fp64 tensor-core step feeds the same Gram kernel
    Hd.set_math_mode(tt.MATH_FP64)
    tt.project(Hd, dev(X), Gd)
    assert relerr(Gd.cpu().numpy(), ref) <= TOL


def test_project_symmetric_shortcut(tt):
    """A handle whose symmetry was verified at build computes only the upper triangle of H_F and mirrors it."""
    import torch
    H, C, _, _ = small_problem(3, 128, 0.4, 2128)
    N = 300
    X = synth.dense_normal(H.M, N, 361)
    ref = oracle.project(C.row_ptr, C.col_idx, C.values, X)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    Gd = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    tt.project(Hd, dev(X), Gd)
    got = Gd.cpu().numpy()
    assert relerr(got, ref) <= TOL
    assert np.array_equal(got, got.T)                        # mirrored: exactly symmetric


def test_project_csr_and_reordered_handles(tt):
    import torch
    H, C, _, _ = small_problem(3, 64, 0.3, 2064)
    perm = synth.permutation(H.M, 77)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // H.b).astype(np.int32)
    N = 90
    X = synth.dense_normal(H.M, N, 341)
    ref = oracle.project(Cp.row_ptr, Cp.col_idx, Cp.values, X)
    Gd = torch.empty(N, N, dtype=torch.float64, device="cuda")
    for lab in (None, labels):                               # generic kernel / reordered tiles
        Hd = tt.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values),
                            subdomain_of_row=None if lab is None else dev(lab))
        assert Hd.info()["reordered"] == (0 if lab is None else 1)
        tt.project(Hd, dev(X), Gd)
        assert relerr(Gd.cpu().numpy(), ref) <= TOL


def test_project_errors(tt):
    import torch
    H, C, _, _ = small_problem(4, 32, 0.0, 1001)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    X = dev(synth.dense_normal(H.M, 8, 351))
    G = torch.empty(8, 8, dtype=torch.float64, device="cuda")
    small = torch.empty(2048, dtype=torch.uint8, device="cuda")
    with pytest.raises(tt.TTDFTError) as e:
        tt.project(Hd, X, G, work=small)
    assert e.value.status_name == "WORKSPACE_TOO_SMALL"
    with pytest.raises(tt.TTDFTError):
        tt.gram(X, X, G, work=small)


def test_project_full_config3_si():
    """BASELINE.json config 3 (M=221,184, N=4,096): a seeded sub-block G[cols, cols] = X_c^T (H X_c) is compared entry by
    entry with the oracle (exact: entry (j,l) depends on columns j and l only), and EVERY entry is covered by the
    Freivalds identity G u = X^T (H (X u)) with the right side evaluated by the oracle's SpMM."""
    import torch
    import paper_2110_15853_b200 as tt
    cfg = synth.CONFIGS["si"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    C = synth.bsr_to_csr_nonzeros(H)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    N = cfg.N
    Xh = np.empty((cfg.M, N))
    synth.dense_normal(cfg.M, N, cfg.seed, synth.STREAM_X, out=Xh)
    Xd = dev(Xh)
    Gd = torch.empty(N, N, dtype=torch.float64, device="cuda")
    tt.project(Hd, Xd, Gd)
    torch.cuda.synchronize()
    got = Gd.cpu().numpy()
    rng = np.random.default_rng(5)
    cols = np.unique(np.concatenate([[0, 63, 64, 127, 128, 2047, 2048, N - 1], rng.integers(0, N, 24)]))
    Xc = np.ascontiguousarray(Xh[:, cols])
    ref = oracle.project(C.row_ptr, C.col_idx, C.values, Xc)
    assert relerr(got[np.ix_(cols, cols)], ref) <= TOL
    assert relerr(got, got.T) <= 1e-13
    u = rng.standard_normal((N, 2))
    z = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, Xh @ u)
    rhs = Xh.T @ z
    assert relerr(got @ u, rhs) <= 1e-11


# ---------------------------------------------------------------- rotation Y = X Q (Algorithm 1 step 5)
@pytest.mark.parametrize("M,K,N,pad", [(2048, 32, 32, 0), (1000, 70, 33, 3), (300, 1, 1, 1), (4113, 130, 257, 5), (77, 300, 64, 0),
                                       (128 * 40, 512, 200, 0)])
def test_rotate_vs_oracle(tt, M, K, N, pad):
    import torch
    X = synth.dense_normal(M, K, 401) * 10.0 ** np.linspace(-6, 6, M)[:, None]      # rows of very different size
    Q = synth.dense_normal(K, N, 402) * 10.0 ** np.linspace(5, -5, N)[None, :]      # columns of very different size
    ref = oracle.rotate(X, Q)
    Xd = torch.zeros(M, K + pad, dtype=torch.float64, device="cuda")
    Qd = torch.zeros(K, N + pad, dtype=torch.float64, device="cuda")
    Xd[:, :K], Qd[:, :N] = dev(X), dev(Q)
    Yd = torch.full((M, N + pad), float("nan"), dtype=torch.float64, device="cuda")
    tt.rotate(Xd[:, :K], Qd[:, :N], Yd[:, :N])
    got = Yd[:, :N].cpu().numpy()
    # entry-wise against the scale of each entry, |x_i| |q_l| (row- and column-scaled fixed point)
    scale = np.outer(np.linalg.norm(X, axis=1), np.linalg.norm(Q, axis=0))
    scale[scale == 0] = 1.0
    assert np.max(np.abs(got - ref) / scale) <= 1e-15 * np.sqrt(K) + 1e-16
    if pad:
        assert torch.isnan(Yd[:, N:]).all()                  # nothing written outside the view
    Y2 = torch.empty(M, N, dtype=torch.float64, device="cuda")
    tt.rotate(Xd[:, :K], Qd[:, :N], Y2)
    assert np.array_equal(Y2.cpu().numpy(), got)             # deterministic


def test_rotate_identity_and_gram_congruence(tt):
    import torch
    M, K = 3000, 96
    X = synth.dense_normal(M, K, 411)
    Xd = dev(X)
    Y = torch.empty(M, K, dtype=torch.float64, device="cuda")
    tt.rotate(Xd, torch.eye(K, dtype=torch.float64, device="cuda"), Y)
    assert relerr(Y.cpu().numpy(), X) <= 1e-15               # Q = I (exact up to the 55-bit rounding of the rows)
    Q = synth.dense_normal(K, K, 412)
    tt.rotate(Xd, dev(Q), Y)
    G, GY = torch.empty(K, K, dtype=torch.float64, device="cuda"), torch.empty(K, K, dtype=torch.float64, device="cuda")
    tt.gram(Xd, Xd, G)
    tt.gram(Y, Y, GY)                                        # (XQ)^T (XQ) = Q^T (X^T X) Q
    assert relerr(GY.cpu().numpy(), Q.T @ G.cpu().numpy() @ Q) <= 1e-12


def test_rotate_full_config3_shape():
    """Config 3's shape (M = 221,184, k = n = 4,096): seeded rows compared entry by entry with the oracle (row i of Y depends on
    row i of X only) and every entry covered by the Freivalds identity Y u = X (Q u)."""
    import torch
    import paper_2110_15853_b200 as tt
    cfg = synth.CONFIGS["si"]
    M, K = cfg.M, cfg.N
    Xh = np.empty((M, K))
    synth.dense_normal(M, K, cfg.seed, synth.STREAM_X, out=Xh)
    Qh = synth.dense_normal(K, K, 421) / np.sqrt(K)
    Xd, Qd = dev(Xh), dev(Qh)
    Yd = torch.empty(M, K, dtype=torch.float64, device="cuda")
    tt.rotate(Xd, Qd, Yd)
    torch.cuda.synchronize()
    rng = np.random.default_rng(6)
    rows = np.unique(np.concatenate([[0, 127, 128, M - 1], rng.integers(0, M, 28)]))
    ref = oracle.rotate(np.ascontiguousarray(Xh[rows]), Qh)
    got_rows = Yd[torch.from_numpy(rows).cuda()].cpu().numpy()
    assert relerr(got_rows, ref) <= TOL
    u = torch.from_numpy(rng.standard_normal((K, 2))).cuda()
    lhs = (Yd @ u).cpu().numpy()
    rhs = Xh @ (Qh @ u.cpu().numpy())
    assert relerr(lhs, rhs) <= 1e-12
