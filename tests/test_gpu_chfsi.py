"""End-to-end check of the composition (paper_2110_15853_b200/chfsi.py): a few passes of Algorithm 1 must
converge to the lowest eigenpairs of H.  Expected values: numpy.linalg.eigh of the dense matrix (a library routine on the CPU,
independent of both the CUDA path and the oracle); residuals are evaluated with the oracle's SpMM."""
import numpy as np
import pytest

import oracle
import synth
from util import small_problem

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("G,b,z,seed,n", [(4, 32, 0.0, 1001, 32), (3, 64, 0.3, 2064, 40)])
def test_chfsi_converges_to_lowest_eigenpairs(G, b, z, seed, n):
    import torch
    import paper_2110_15853_b200 as tt
    from paper_2110_15853_b200.chfsi import chfsi
    H, C, _, (a0, bb) = small_problem(G, b, z, seed)
    dense = np.zeros((H.M, H.M))
    rows = np.repeat(np.arange(H.M), np.diff(C.row_ptr))
    dense[rows, C.col_idx] = C.values
    lam_true = np.linalg.eigvalsh(dense)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    X = dev(synth.dense_normal(H.M, n, 601))
    Psi, lam = chfsi(Hd, X, m=12, b=bb, a0=a0, iterations=15)
    lam = lam.cpu().numpy()
    psi = Psi.cpu().numpy()
    nconv = n // 2                                           # the top of the block converges last (small gaps): judge the lower half
    assert np.max(np.abs(lam[:nconv] - lam_true[:nconv])) <= 1e-8 * np.abs(lam_true).max()
    assert np.linalg.norm(psi.T @ psi - np.eye(n)) <= 1e-12 * n
    R = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, psi) - psi * lam[None, :]
    assert np.max(np.linalg.norm(R[:, :nconv], axis=0)) <= 1e-6 * np.abs(lam_true).max()
