"""A0, HYBRID input: the paper's own layout (Sec. 4.1, Fig. 3: "the diagonal blocks and the off-diagonal blocks of
the Hamiltonian matrix are stored as dense and sparse matrices") handed to ttdft_h_build as (dense diagonal blocks, CSR of the
rest).  The library forms the union -- tiles when the subdomain labels are usable, one CSR otherwise -- and every product must
equal the CPU oracle's on the plain CSR of the same matrix."""
import numpy as np
import pytest

import oracle
import synth
from util import bounds_for, relerr, small_problem, worst_col_relerr

pytestmark = pytest.mark.gpu

TOL_SPMM = 1e-12
TOL_FILTER = 1e-10


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2110_15853_b200 as t
    assert torch.cuda.is_available()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def build_hybrid(t, C, D, labels=None, flags=0):
    diag, od = synth.split_hybrid(C, D)
    return t.h_build_hybrid(C.M, D, dev(diag), dev(od.row_ptr), dev(od.col_idx), dev(od.values),
                            subdomain_of_row=None if labels is None else dev(labels), flags=flags), diag, od


# D: a multiple of the tile size, not a multiple (blocks cut through subdomains), larger than M / 2 (ragged last block), M itself
@pytest.mark.parametrize("G,b,z,D", [(3, 64, 0.3, 256), (3, 64, 0.3, 200), (2, 128, 0.4, 700), (2, 96, 0.4, 768), (4, 32, 0.0, 96)])
def test_hybrid_with_labels_becomes_tiles(tt, G, b, z, D):
    H, C, _, _ = small_problem(G, b, z, 5100 + b)
    labels = (np.arange(H.M) // b).astype(np.int32)
    Hd, diag, od = build_hybrid(tt, C, D, labels, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    assert od.nnz < C.nnz and np.count_nonzero(diag) + od.nnz == C.nnz        # the split really has two parts
    info = Hd.info()
    assert info["kernel"] == 1 and info["block"] == b
    assert info["nblocks"] == H.nblocks                      # tiles exactly where the generator put them
    N = 70
    X = synth.dense_normal(H.M, N, 91)
    Y0 = synth.dense_normal(H.M, N, 92)
    ref = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.25, X, -0.5, Y0.copy())
    for mode in (tt.MATH_FP64, tt.MATH_I8X7):
        if mode != tt.MATH_FP64 and b < 64:
            continue
        Hd.set_math_mode(mode)
        Y = dev(Y0)
        tt.spmm(Hd, 1.25, dev(X), -0.5, Y, use_work=True)
        assert relerr(Y.cpu().numpy(), ref) <= TOL_SPMM


def test_hybrid_tiles_equal_csr_build_bit_for_bit(tt):
    """The same matrix through the CSR and the HYBRID description gives the same tiles, hence identical results."""
    import torch
    H, C, _, (a0, bb) = small_problem(3, 64, 0.3, 5200)
    labels = (np.arange(H.M) // 64).astype(np.int32)
    Hh, _, _ = build_hybrid(tt, C, 320, labels)
    Hc = tt.h_build_csr(C.M, dev(C.row_ptr), dev(C.col_idx), dev(C.values), subdomain_of_row=dev(labels))
    a, b_, a0_ = bounds_for(a0, bb, 48, H.M)
    X = dev(synth.dense_normal(H.M, 48, 93))
    Yh, Yc = torch.empty_like(X), torch.empty_like(X)
    tt.cheb_filter(Hh, X, Yh, 9, a, b_, a0_)
    tt.cheb_filter(Hc, X, Yc, 9, a, b_, a0_)
    assert torch.equal(Yh, Yc)


@pytest.mark.parametrize("D", [1, 37, 300])
def test_hybrid_without_labels_becomes_one_csr(tt, D):
    H, C, _, (a0, bb) = small_problem(3, 32, 0.5, 5300)
    Hd, diag, od = build_hybrid(tt, C, D, None, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    info = Hd.info()
    assert info["kernel"] == 0 and info["nnz_stored"] == C.nnz           # zeros of the dense blocks are not stored
    N = 33
    X = synth.dense_normal(H.M, N, 94)
    Y0 = synth.dense_normal(H.M, N, 95)
    ref = oracle.spmm(C.row_ptr, C.col_idx, C.values, -2.0, X, 0.75, Y0.copy())
    Y = dev(Y0)
    tt.spmm(Hd, -2.0, dev(X), 0.75, Y)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_SPMM
    m = 8
    a, b_, a0_ = bounds_for(a0, bb, N, H.M)
    reff = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, b_, a0_)
    import torch
    Yf = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Yf, m, a, b_, a0_)
    assert worst_col_relerr(Yf.cpu().numpy(), reff) <= TOL_FILTER


def test_hybrid_permuted_rows_with_labels(tt):
    """Rows in any order (label layout 2): the dense blocks then cut across subdomains arbitrarily."""
    b = 64
    H, C, _, _ = small_problem(3, b, 0.3, 5400)
    perm = synth.permutation(H.M, 5450)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // b).astype(np.int32)
    Hd, _, _ = build_hybrid(tt, Cp, 500, labels, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    info = Hd.info()
    assert info["kernel"] == 1 and info["reordered"] == 1 and info["nblocks"] == H.nblocks
    N = 40
    X = synth.dense_normal(H.M, N, 96)
    ref = oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, X, 0.0, np.zeros_like(X))
    import torch
    Y = torch.zeros(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_SPMM


def test_hybrid_validation(tt):
    H, C, _, _ = small_problem(2, 32, 0.3, 5500)
    D = 64
    diag, od = synth.split_hybrid(C, D)
    # an off-diagonal entry inside a diagonal block: the plain CSR of the whole matrix as the "off-diagonal" part
    with pytest.raises(tt.TTDFTError) as e:
        tt.h_build_hybrid(C.M, D, dev(diag), dev(C.row_ptr), dev(C.col_idx), dev(C.values), flags=tt.CHECK_SORTED)
    assert e.value.status_name == "INVALID_ARG"
    # a dense block that is not symmetric
    bad = diag.copy()
    bad[0, 0, 1] += 1.0
    with pytest.raises(tt.TTDFTError) as e:
        tt.h_build_hybrid(C.M, D, dev(bad), dev(od.row_ptr), dev(od.col_idx), dev(od.values), flags=tt.CHECK_SYMMETRY)
    assert e.value.status_name == "NOT_SYMMETRIC"
    # diag_block out of range, diag_values missing
    for Dbad in (0, C.M + 1):
        with pytest.raises(tt.TTDFTError) as e:
            tt.h_build(tt.api.FMT_HYBRID, C.M, 0, dev(od.row_ptr), dev(od.col_idx), dev(od.values), diag_values=dev(diag).reshape(-1),
                       diag_block=Dbad)
        assert e.value.status_name == "INVALID_ARG"
    with pytest.raises(tt.TTDFTError) as e:
        tt.h_build(tt.api.FMT_HYBRID, C.M, 0, dev(od.row_ptr), dev(od.col_idx), dev(od.values), diag_values=None, diag_block=D)
    assert e.value.status_name == "INVALID_ARG"
