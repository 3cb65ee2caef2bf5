"""ttdft_cheb_step_static: the fused recurrence step with the library's own static device scratch, for callers
that cannot allocate device memory.  Its output must equal the existing path's (ttdft_cheb_step_ws on caller scratch) -- the two
run the same kernels, so the comparison is bit for bit, and both are checked against the CPU oracle at the tolerance of the other
step tests -- on two calls in a row with different inputs (the shared scratch keeps the first call's contents).
Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import oracle
import synth
from util import relerr, small_problem

pytestmark = pytest.mark.gpu

TOL_SPMM = 1e-12


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2110_15853_b200 as t
    assert torch.cuda.is_available()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("b,mode", [(128, "I8X7"), (64, "I8X7"), (128, "I8"), (64, "FP64")])
def test_static_scratch_step_equals_ws_step_two_calls(tt, b, mode):
    import torch
    H, C, _, _ = small_problem(3, b, 0.3, 7100 + b)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    Hd.set_math_mode(getattr(tt, "MATH_" + mode))
    need = tt.step_work_bytes(Hd, 200)
    assert need <= tt.STATIC_SCRATCH_BYTES
    if mode != "FP64":
        assert need > 0                                    # the int8 modes really use the scratch
    # two calls in a row: different widths (200 columns = ragged last tile, then 70), values and scalars, so anything the first
    # call left in the shared scratch is wrong for the second
    for N, seed, (al, c, be) in ((200, 11, (0.7, -1.3, -0.4)), (70, 12, (-1.1, 0.6, 0.9))):
        X = synth.dense_normal(H.M, N, seed)
        Z = synth.dense_normal(H.M, N, seed + 100)
        ref = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, al, c, be, X, Z)
        Xd, Zd = dev(X), dev(Z)
        Ows = torch.full((H.M, N), float("nan"), dtype=torch.float64, device="cuda")
        Ost = torch.full((H.M, N), float("nan"), dtype=torch.float64, device="cuda")
        tt.cheb_step(Hd, al, c, be, Xd, Zd, Ows, use_work=True)          # the existing path: caller scratch
        tt.cheb_step_static(Hd, al, c, be, Xd, Zd, Ost)                  # the new one: static scratch
        torch.cuda.synchronize()
        assert relerr(Ows.cpu().numpy(), ref) <= TOL_SPMM
        assert relerr(Ost.cpu().numpy(), ref) <= TOL_SPMM
        assert relerr(Ost.cpu().numpy(), Ows.cpu().numpy()) <= TOL_SPMM
        assert torch.equal(Ost, Ows)                                     # same kernels, same order of operations
    # the first step of a filter: no Y_{k-1}
    X = synth.dense_normal(H.M, 33, 13)
    Xd = dev(X)
    O1 = torch.empty(H.M, 33, dtype=torch.float64, device="cuda")
    O2 = torch.empty_like(O1)
    tt.cheb_step(Hd, 0.5, 2.0, 0.0, Xd, None, O1, use_work=True)
    tt.cheb_step_static(Hd, 0.5, 2.0, 0.0, Xd, None, O2)
    assert torch.equal(O1, O2)
    assert relerr(O2.cpu().numpy(), oracle.cheb_step(C.row_ptr, C.col_idx, C.values, 0.5, 2.0, 0.0, X, None)) <= TOL_SPMM


def test_static_scratch_reordered_handle(tt):
    """A handle built from permuted rows + labels takes two panels in tile order from the scratch as well."""
    import torch
    b = 64
    H, C, _, _ = small_problem(3, b, 0.3, 7300)
    perm = synth.permutation(H.M, 7350)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // b).astype(np.int32)
    Hd = tt.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values), subdomain_of_row=dev(labels))
    assert Hd.info()["reordered"] == 1
    for N, seed in ((96, 21), (40, 22)):
        X = synth.dense_normal(H.M, N, seed)
        Z = synth.dense_normal(H.M, N, seed + 100)
        Xd, Zd = dev(X), dev(Z)
        O1 = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
        O2 = torch.empty_like(O1)
        tt.cheb_step(Hd, 1.2, 0.3, -0.7, Xd, Zd, O1, use_work=True)
        tt.cheb_step_static(Hd, 1.2, 0.3, -0.7, Xd, Zd, O2)
        assert torch.equal(O1, O2)
        assert relerr(O2.cpu().numpy(), oracle.cheb_step(Cp.row_ptr, Cp.col_idx, Cp.values, 1.2, 0.3, -0.7, X, Z)) <= TOL_SPMM


def test_static_scratch_rejects_steps_beyond_its_size(tt):
    import torch
    H, C, _, _ = small_problem(3, 128, 0.3, 7400)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    Hd.set_math_mode(tt.MATH_I8X7)
    N = 2048
    while tt.step_work_bytes(Hd, N) <= tt.STATIC_SCRATCH_BYTES:
        N *= 2
    X = torch.zeros(H.M, N, dtype=torch.float64, device="cuda")
    O = torch.full((H.M, N), 7.0, dtype=torch.float64, device="cuda")
    n0 = tt.launch_count()
    with pytest.raises(tt.TTDFTError) as e:
        tt.cheb_step_static(Hd, 1.0, 0.0, 0.0, X, None, O)
    assert e.value.status_name == "WORKSPACE_TOO_SMALL"
    assert "static scratch" in tt.last_error()
    assert tt.launch_count() == n0                         # nothing was launched
    assert bool((O == 7.0).all())
    # the largest width that fits still runs
    while tt.step_work_bytes(Hd, N) > tt.STATIC_SCRATCH_BYTES:
        N -= 64
    X = dev(synth.dense_normal(H.M, N, 31))
    O = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_step_static(Hd, 1.0, 0.0, 0.0, X, None, O)
    ref_cols = [0, N // 2, N - 1]
    Xs = np.ascontiguousarray(X.cpu().numpy()[:, ref_cols])
    ref = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, 1.0, 0.0, 0.0, Xs, None)
    assert relerr(O.cpu().numpy()[:, ref_cols], ref) <= TOL_SPMM
