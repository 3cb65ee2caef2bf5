"""GPU parity of the orthonormalisation X_F = Orth(X) (Algorithm 1 step 2, L230 "Gram-Schmidt
orthogonalization procedure"): ttdft_orthonormalize (Cholesky-QR on the tensor-core Gram and rotation kernels) against the
CPU oracle's Gram-Schmidt.  For full-rank X both compute THE Q of the QR factorisation with a positive diagonal of R, so
they are compared entry by entry; the tolerance grows with cond(X) because Q itself is that sensitive to rounding."""
import numpy as np
import pytest

import oracle
import synth
from util import relerr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2110_15853_b200 as t
    assert torch.cuda.is_available()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def conditioned(M, n, cond, seed):
    X = synth.dense_normal(M, n, seed)
    if cond > 1.0:
        U, _, Vt = np.linalg.svd(X, full_matrices=False)
        X = np.ascontiguousarray((U * np.logspace(0, -np.log10(cond), n)) @ Vt)
    return X


@pytest.mark.parametrize("M,n,cond,pad", [(2048, 32, 1.0, 0), (1000, 70, 1.0, 3), (4113, 130, 1e3, 0), (300, 1, 1.0, 1),
                                          (5000, 257, 1e5, 5), (128, 128, 1.0, 0),
                                          (3000, 449, 1e2, 1), (2500, 320, 1.0, 0)])     # 8 and 5 column tiles: the triangular tile limit of the rotation
def test_orthonormalize_vs_gram_schmidt(tt, M, n, cond, pad):
    import torch
    X = conditioned(M, n, cond, 501)
    ref = oracle.orthonormalize(X)
    Xd = torch.zeros(M, n + pad, dtype=torch.float64, device="cuda")
    Xd[:, :n] = dev(X)
    Yd = torch.full((M, n + pad), float("nan"), dtype=torch.float64, device="cuda")
    tt.orthonormalize(Xd[:, :n], Yd[:, :n])                       # Cholesky-QR2
    got = Yd[:, :n].cpu().numpy()
    assert relerr(got, ref) <= 1e-13 * max(cond, 10.0)
    assert np.linalg.norm(got.T @ got - np.eye(n)) <= 1e-13 * np.sqrt(n)     # orthonormal to rounding level
    R = got.T @ X
    assert np.linalg.norm(np.tril(R, -1)) <= 1e-12 * np.linalg.norm(R) and np.all(np.diag(R) > 0)
    assert np.linalg.norm(got @ R - X) <= 1e-12 * np.linalg.norm(X)          # same span
    if pad:
        assert torch.isnan(Yd[:, n:]).all()
    assert np.array_equal(Xd[:, :n].cpu().numpy(), X)             # X untouched


def test_single_pass_and_breakdown(tt):
    import torch
    M, n = 3000, 64
    X = conditioned(M, n, 1e4, 511)
    Xd = dev(X)
    Y1 = torch.empty_like(Xd)
    tt.orthonormalize(Xd, Y1, passes=1)                          # plain Cholesky-QR: orthogonality ~ cond^2 * eps
    q1 = Y1.cpu().numpy()
    d1 = np.linalg.norm(q1.T @ q1 - np.eye(n))
    assert 1e-13 < d1 <= 1e-6
    Y2 = torch.empty_like(Xd)
    tt.orthonormalize(Xd, Y2, passes=2)
    q2 = Y2.cpu().numpy()
    assert np.linalg.norm(q2.T @ q2 - np.eye(n)) <= 1e-13 * np.sqrt(n)
    # dependent columns: X^T X is singular -> TTDFT_ERR_BREAKDOWN, not garbage
    Xb = X.copy()
    Xb[:, 7] = Xb[:, 3]
    with pytest.raises(tt.TTDFTError) as e:
        tt.orthonormalize(dev(Xb), Y2)
    assert e.value.status_name == "BREAKDOWN"
    with pytest.raises(tt.TTDFTError):
        tt.orthonormalize(Xd, Xd)                                # overlap


def test_orthonormalize_async_no_sync_and_graph_capture(tt):
    """ttdft_orthonormalize_async: the same result bit for bit, the breakdown flag left on the device (0 per pass; non-zero for
    dependent columns, where the call still runs to the end), and the call captures into a CUDA graph (no synchronisation inside)."""
    import torch
    M, n = 3000, 200
    X = conditioned(M, n, 1e3, 521)
    Xd = dev(X)
    Y1 = torch.empty_like(Xd)
    tt.orthonormalize(Xd, Y1, passes=2)
    Y2 = torch.full_like(Xd, float("nan"))
    st = torch.full((2,), -1, dtype=torch.int32, device="cuda")
    work = torch.empty(tt.orthonormalize_work_bytes(M, n, 2) + 1024, dtype=torch.uint8, device="cuda")
    tt.orthonormalize_async(Xd, Y2, st, passes=2, work=work)
    assert torch.equal(Y1, Y2) and st.tolist() == [0, 0]
    assert relerr(Y2.cpu().numpy(), oracle.orthonormalize(X)) <= 1e-13 * 1e3
    # captured into a graph and replayed on new contents of the same buffers
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            tt.orthonormalize_async(Xd, Y2, st, passes=2, work=work, stream=s)
    torch.cuda.current_stream().wait_stream(s)
    X2 = conditioned(M, n, 10.0, 522)
    Xd.copy_(dev(X2))
    Y2.fill_(float("nan"))
    st.fill_(-1)
    g.replay()
    torch.cuda.synchronize()
    assert st.tolist() == [0, 0]
    assert relerr(Y2.cpu().numpy(), oracle.orthonormalize(X2)) <= 1e-12
    # dependent columns (the matrix of test_single_pass_and_breakdown): no error status from the call, the flag on the device says
    # which pivot broke down -- the same one the synchronising call reports
    Xb = conditioned(3000, 64, 1e4, 511)
    Xb[:, 7] = Xb[:, 3]
    Xbd = dev(Xb)
    Yb = torch.empty_like(Xbd)
    st.fill_(-1)
    tt.orthonormalize_async(Xbd, Yb, st, passes=2)
    torch.cuda.synchronize()
    flags = st.tolist()
    assert all(f >= 0 for f in flags) and any(f > 0 for f in flags)
    first = next(f for f in flags if f > 0)
    with pytest.raises(tt.TTDFTError) as e:
        tt.orthonormalize(Xbd, Yb)
    assert e.value.status_name == "BREAKDOWN" and ("(pivot %d)" % (first - 1)) in tt.last_error()
    with pytest.raises(TypeError):
        tt.orthonormalize_async(Xd, Y2, torch.zeros(1, dtype=torch.int32, device="cuda"), passes=2)      # needs one entry per pass


def test_orthonormalize_full_config3_shape():
    """Config 3's shape (M = 221,184, n = 4,096): a leading block of columns is compared with the oracle's Gram-Schmidt (column j of
    Q depends on columns 0..j of X only), orthonormality is checked on a seeded sample of column pairs through the oracle's Gram
    product, and the span through X = Q (Q^T X) on sampled columns."""
    import torch
    import paper_2110_15853_b200 as tt
    cfg = synth.CONFIGS["si"]
    M, n = cfg.M, cfg.N
    Xh = np.empty((M, n))
    synth.dense_normal(M, n, cfg.seed, synth.STREAM_X, out=Xh)
    Xd = dev(Xh)
    Yd = torch.empty_like(Xd)
    tt.orthonormalize(Xd, Yd)
    torch.cuda.synchronize()
    lead = 24
    ref = oracle.orthonormalize(np.ascontiguousarray(Xh[:, :lead]))
    assert relerr(Yd[:, :lead].cpu().numpy(), ref) <= 1e-12
    rng = np.random.default_rng(7)
    cols = np.unique(np.concatenate([[0, 63, 64, 127, 128, n - 1], rng.integers(0, n, 26)]))
    Qc = np.ascontiguousarray(Yd[:, torch.from_numpy(cols).cuda()].cpu().numpy())
    G = oracle.gram(Qc, Qc)
    assert np.linalg.norm(G - np.eye(len(cols))) <= 1e-13 * len(cols)
