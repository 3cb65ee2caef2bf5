"""Seeded random differential test of the filter entry points against the CPU oracle: tile size, sparsity, column count (ragged),
leading-dimension padding, panel width, degree, in-place / out-of-place, math mode and input layout (BSR, CSR with labels in any
row order) are all drawn at random; every case must meet north_star's tolerance."""
import numpy as np
import pytest

import oracle
import synth
from util import bounds_for, relerr, small_problem, worst_col_relerr

pytestmark = pytest.mark.gpu

CASES = list(range(40))


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("case", CASES)
def test_random_filter_case(case):
    import torch
    import paper_2110_15853_b200 as tt
    rng = np.random.default_rng(7000 + case)
    G, b = [(2, 128), (3, 64), (2, 96), (3, 32), (2, 64), (3, 96)][rng.integers(0, 6)]
    z = float(rng.choice([0.0, 0.3, 0.6]))
    H, C, _, (a0, bb) = small_problem(G, b, z, 4000 + b + G)
    N = int(rng.choice([1, 7, 31, 64, 65, 100, 129, 200]))
    pad = int(rng.choice([0, 0, 1, 3, 8]))
    m = int(rng.integers(0, 13))
    panel = int(rng.choice([0, 0, 16, 33, 64, 100]))
    inplace = bool(rng.integers(0, 2))
    layout = str(rng.choice(["bsr", "csr+labels", "csr+permuted-labels"]))
    mode = str(rng.choice(["auto", "fp64", "i8", "i8x7"]))
    a, bb, a0 = bounds_for(a0, bb, max(N, 8), H.M, wide=bool(rng.integers(0, 2)))
    X = synth.dense_normal(H.M, N, 8000 + case)
    if layout == "bsr":
        Cuse = C
        Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    elif layout == "csr+labels":
        Cuse = C
        labels = (np.arange(H.M) // b).astype(np.int32)
        Hd = tt.h_build_csr(C.M, dev(C.row_ptr), dev(C.col_idx), dev(C.values), subdomain_of_row=dev(labels))
    else:
        perm = synth.permutation(H.M, 9000 + case)
        Cuse = synth.permute_csr(C, perm)
        labels = np.empty(H.M, np.int32)
        labels[perm] = (np.arange(H.M) // b).astype(np.int32)
        Hd = tt.h_build_csr(Cuse.M, dev(Cuse.row_ptr), dev(Cuse.col_idx), dev(Cuse.values), subdomain_of_row=dev(labels))
        assert Hd.info()["reordered"] == 1
    assert Hd.info()["kernel"] == 1
    if mode != "auto" and not (mode in ("i8", "i8x7") and Hd.info()["i8_planes"] == 0):
        Hd.set_math_mode({"fp64": tt.MATH_FP64, "i8": tt.MATH_I8, "i8x7": tt.MATH_I8X7}[mode])
    ref = oracle.cheb_filter(Cuse.row_ptr, Cuse.col_idx, Cuse.values, X, m, a, bb, a0)
    Xd = torch.zeros(H.M, N + pad, dtype=torch.float64, device="cuda")
    Xd[:, :N] = dev(X)
    if inplace:
        Yd = Xd
    else:
        Yd = torch.full((H.M, N + pad), float("nan"), dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, Xd[:, :N], Yd[:, :N], m, a, bb, a0, panel_cols=panel)
    got = Yd[:, :N].cpu().numpy()
    desc = f"G={G} b={b} z={z} N={N} pad={pad} m={m} panel={panel} inplace={inplace} layout={layout} mode={mode}"
    assert relerr(got, ref) <= 1e-10, desc
    assert worst_col_relerr(got, ref) <= 1e-9, desc
    if pad and not inplace:
        assert torch.isnan(Yd[:, N:]).all(), desc
    if pad and inplace:
        assert (Yd[:, N:] == 0).all(), desc
