"""GPU parity of ttdft_lanczos_bounds (the bounds Algorithm 1 takes as inputs; DESIGN.md
reading #5) against the CPU oracle's Lanczos (pinned by P6) and against numpy's dense eigenvalues."""
import numpy as np
import pytest

import oracle
import synth
from util import small_problem

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("G,b,z,seed,layout", [(4, 32, 0.0, 1001, "bsr"), (3, 64, 0.3, 2064, "bsr"), (3, 64, 0.3, 2064, "csr"),
                                               (2, 128, 0.4, 2128, "csr+permuted-labels")])
def test_lanczos_bounds_vs_oracle(G, b, z, seed, layout):
    import paper_2110_15853_b200 as tt
    H, C, _, _ = small_problem(G, b, z, seed)
    v0 = synth.dense_normal(H.M, 1, seed, synth.STREAM_V0).reshape(-1)
    Cuse, v0use = C, v0
    if layout == "bsr":
        Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    elif layout == "csr":
        Hd = tt.h_build_csr(C.M, dev(C.row_ptr), dev(C.col_idx), dev(C.values))
    else:
        perm = synth.permutation(H.M, seed + 9)
        Cuse = synth.permute_csr(C, perm)
        labels = np.empty(H.M, np.int32)
        labels[perm] = (np.arange(H.M) // b).astype(np.int32)
        v0use = synth.permute_rows(v0.reshape(-1, 1), perm).reshape(-1)
        Hd = tt.h_build_csr(Cuse.M, dev(Cuse.row_ptr), dev(Cuse.col_idx), dev(Cuse.values), subdomain_of_row=dev(labels))
    k = 30
    a0_ref, b_ref, info = oracle.lanczos_bounds(Cuse.row_ptr, Cuse.col_idx, Cuse.values, v0use, k)
    a0, bb, theta = tt.lanczos_bounds(Hd, dev(v0use), k)
    width = b_ref - a0_ref
    assert len(theta) == len(info["theta"])
    assert abs(a0 - a0_ref) <= 1e-9 * width and abs(bb - b_ref) <= 1e-9 * width
    assert np.max(np.abs(np.array(theta) - info["theta"])) <= 1e-8 * width
    dense = np.zeros((H.M, H.M))
    rows = np.repeat(np.arange(H.M), np.diff(C.row_ptr))
    dense[rows, C.col_idx] = C.values
    lam = np.linalg.eigvalsh(dense)
    assert a0 <= lam[0] + 1e-12 * width and bb >= lam[-1] - 1e-12 * width      # valid bounds of the true spectrum


def test_lanczos_errors_and_invariant_subspace():
    import torch
    import paper_2110_15853_b200 as tt
    H, C, _, _ = small_problem(4, 32, 0.0, 1001)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    with pytest.raises(tt.TTDFTError):
        tt.lanczos_bounds(Hd, torch.zeros(H.M, dtype=torch.float64, device="cuda"), 10)   # zero start vector
    with pytest.raises(tt.TTDFTError):
        tt.lanczos_bounds(Hd, dev(np.ones(H.M)), 65)                                      # k too large
    # H = diag(d) as 32 x 32 tiles: a start vector with 3 non-zero entries spans an invariant subspace of dimension 3
    M, b = 128, 32
    d = np.linspace(1.0, 9.0, M)
    vals = np.zeros((4, b, b))
    for I in range(4):
        vals[I][np.arange(b), np.arange(b)] = d[I * b:(I + 1) * b]
    Hdiag = tt.h_build_bsr(M, b, dev(np.arange(5, dtype=np.int32)), dev(np.arange(4, dtype=np.int32)), dev(vals))
    v0 = np.zeros(M)
    v0[[3, 40, 100]] = [1.0, 2.0, -1.0]
    a0, bb, theta = tt.lanczos_bounds(Hdiag, dev(v0), 10)
    # beta_3 is ~1e-16, not exactly 0, so the recurrence goes on from rounding noise (as the oracle's would): the three
    # eigenvalues of the invariant subspace are found to full accuracy and the bounds stay inside the true spectrum
    want = d[[3, 40, 100]]
    assert all(np.min(np.abs(np.array(theta) - w)) <= 1e-9 for w in want)
    assert d[0] - 1e-9 <= a0 <= d[3] + 1e-9 and d[100] - 1e-9 <= bb <= d[-1] + 1e-9
