"""Boundary behaviour of the C ABI on a GPU (include/ttdft.h conventions): scratch checks on reordered handles, validation before
any kernel consumes the indices, column views of one buffer as non-overlapping operands.  Expected values: the CPU oracle."""
import ctypes

import numpy as np
import pytest

import oracle
import synth
from util import bounds_for, relerr, small_problem

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


def permuted(G, b, z, seed):
    H, C, _, (a0, bb) = small_problem(G, b, z, seed)
    perm = synth.permutation(H.M, seed + 50)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // b).astype(np.int32)
    return H, Cp, labels, (a0, bb)


@pytest.mark.parametrize("b", [32, 64])
def test_reordered_handle_m1_needs_work(tt, b):
    """A handle whose rows were regrouped by label steps through the scratch panel even for m = 1 out of place: a NULL / short
    `work` must be refused (TTDFT_ERR_WORKSPACE_TOO_SMALL), not written through."""
    import torch
    from paper_2110_15853_b200 import api
    H, Cp, labels, (a0, bb) = permuted(3, b, 0.3, 5100 + b)
    Hd = tt.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values), subdomain_of_row=dev(labels))
    assert Hd.info()["reordered"] == 1
    Hd.set_math_mode(tt.MATH_FP64)
    N = 24
    a, bb, a0 = bounds_for(a0, bb, N, H.M)
    X = synth.dense_normal(H.M, N, 9)
    Xd = dev(X)
    Yd = torch.full((H.M, N), float("nan"), dtype=torch.float64, device="cuda")
    L = api._load()
    st = L.ttdft_cheb_filter(Hd.handle, Xd.data_ptr(), N, Yd.data_ptr(), N, N, 1, a, bb, a0, 0, None, 0, None)
    assert st == 3, (st, tt.last_error())                    # TTDFT_ERR_WORKSPACE_TOO_SMALL
    torch.cuda.synchronize()                                 # no sticky error: the context is still usable
    assert torch.isnan(Yd).all()                             # outputs untouched on error
    tt.cheb_filter(Hd, Xd, Yd, 1, a, bb, a0)                 # with the scratch the binding allocates
    ref = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, 1, a, bb, a0)
    assert relerr(Yd.cpu().numpy(), ref) <= 1e-12


def test_invalid_indices_are_reported_not_faulted(tt):
    """TTDFT_CHECK_SORTED runs before the label analysis / tile count read the indices; without the flag the conversion skips
    invalid entries.  Either way the CUDA context survives."""
    import torch
    H, Cp, labels, _ = permuted(3, 64, 0.3, 5200)
    good = Cp.col_idx.copy()
    for how in ("huge", "negative", "unsorted", "rowptr"):
        ci, rp = good.copy(), Cp.row_ptr.copy()
        if how == "huge":
            ci[12345] = 2**30
        elif how == "negative":
            ci[777] = -5
        elif how == "unsorted":
            e = int(rp[40])
            ci[e], ci[e + 1] = ci[e + 1], ci[e]
        else:
            rp[17] = rp[18] + 3                                 # row 17 would end before it starts
        for lab in (dev(labels), None):
            with pytest.raises(tt.TTDFTError) as err:
                tt.h_build_csr(Cp.M, dev(rp), dev(ci), dev(Cp.values), subdomain_of_row=lab, flags=tt.CHECK_SORTED)
            assert err.value.status_name == "INVALID_ARG"
            torch.cuda.synchronize()
        if how in ("huge", "negative"):
            # no check requested: sizing and conversion must not fault on the bad column (the result is undefined)
            n = tt.h_storage_bytes(0, Cp.M, 0, dev(rp), dev(ci), dev(Cp.values), subdomain_of_row=dev(labels))
            assert n > 0
            tt.h_build_csr(Cp.M, dev(rp), dev(ci), dev(Cp.values), subdomain_of_row=dev(labels))
            torch.cuda.synchronize()
    # the context is intact: the valid matrix still builds and multiplies
    Hd = tt.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(good), dev(Cp.values), subdomain_of_row=dev(labels),
                        flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    X = synth.dense_normal(H.M, 16, 3)
    Y = torch.empty(H.M, 16, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, good, Cp.values, 1.0, X)) <= 1e-12


def test_h_build_on_a_non_blocking_stream(tt):
    """Every builder kernel runs on the caller's stream: inputs produced on a non-blocking stream just before the call are seen."""
    import torch
    H, Cp, labels, _ = permuted(3, 64, 0.3, 5300)
    st = torch.cuda.Stream()
    host = [torch.from_numpy(x).pin_memory() for x in (Cp.row_ptr, Cp.col_idx, Cp.values, labels)]
    X = synth.dense_normal(H.M, 8, 5)
    with torch.cuda.stream(st):
        rp, ci, va, lab = (h.to("cuda", non_blocking=True) for h in host)
        Hd = tt.h_build_csr(Cp.M, rp, ci, va, subdomain_of_row=lab, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY, stream=st)
        Xd = dev(X)
        Y = torch.empty(H.M, 8, dtype=torch.float64, device="cuda")
        tt.spmm(Hd, 1.0, Xd, 0.0, Y, stream=st, use_work=True)
    st.synchronize()
    assert Hd.info()["reordered"] == 1
    assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, X)) <= 1e-12


@pytest.mark.parametrize("b", [32, 128])
def test_column_views_of_one_buffer_do_not_overlap(tt, b):
    """X = B[:, :n] and Y = B[:, n:2n] share a leading dimension and no element: every out-of-place call must accept them;
    views that do share columns are still refused."""
    import torch
    H, C, (rp, col, val), (a0, bb) = small_problem(3, b, 0.4, 5400 + b)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    n, m = 40, 4
    a, bb, a0 = bounds_for(a0, bb, n, H.M)
    X = synth.dense_normal(H.M, n, 7)
    B = torch.full((H.M, 2 * n + 6), float("nan"), dtype=torch.float64, device="cuda")
    B[:, :n] = dev(X)
    tt.spmm(Hd, 1.0, B[:, :n], 0.0, B[:, n:2 * n])
    assert relerr(B[:, n:2 * n].cpu().numpy(), oracle.spmm(rp, col, val, 1.0, X)) <= 1e-12
    tt.cheb_filter(Hd, B[:, :n], B[:, n:2 * n], m, a, bb, a0)
    assert relerr(B[:, n:2 * n].cpu().numpy(), oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)) <= 1e-10
    assert torch.isnan(B[:, 2 * n:]).all() and torch.equal(B[:, :n], dev(X))
    Y = torch.empty(H.M, n, dtype=torch.float64, device="cuda")
    tt.cheb_step(Hd, 0.2, 9.0, 0.0, B[:, :n], None, B[:, n:2 * n])
    with pytest.raises(tt.TTDFTError) as err:
        tt.spmm(Hd, 1.0, B[:, :n], 0.0, B[:, n - 1:2 * n - 1])       # one shared column
    assert err.value.status_name == "INVALID_ARG"
    with pytest.raises(tt.TTDFTError):
        tt.spmm(Hd, 1.0, B[:, 10:10 + n], 0.0, B[:, :n])
    del Y
