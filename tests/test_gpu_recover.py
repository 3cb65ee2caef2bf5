"""A0 without labels (SURVEY.md 8(a) A0, 8(f)-4 "locality recovery for unhinted CSR"; reading #18): the library recovers
the subdomain of every row of a symmetrically permuted CSR from its sparsity pattern.  Integer work, so the bar is bit-exact:
the labels equal the oracle's (oracle/recover.py) and the generator's planted partition; the handle built from them runs the
tile kernels and the filter still matches the oracle on the permuted CSR in the CALLER's row order."""
import numpy as np
import pytest

import oracle
import synth
from oracle.recover import recover_subdomains as oracle_recover
from util import bounds_for, relerr, small_problem, worst_col_relerr

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


def canonical(labels):
    labels = np.asarray(labels)
    first = np.full(int(labels.max()) + 1, -1, np.int64)
    for i in range(len(labels) - 1, -1, -1):
        first[labels[i]] = i
    return first[labels]


def planted(G, b, z, seed):
    H = synth.hamiltonian_bsr(G, b, z, seed)
    C = synth.bsr_to_csr_nonzeros(H)
    perm = synth.permutation(H.M, seed + 50)
    Cp = synth.permute_csr(C, perm)
    truth = np.empty(H.M, np.int32)
    truth[perm] = (np.arange(H.M) // b).astype(np.int32)
    return H, C, Cp, truth


@pytest.mark.parametrize("G,b,z", [(3, 32, 0.0), (3, 32, 0.4), (3, 64, 0.3), (4, 32, 0.4), (3, 96, 0.4), (5, 8, 0.3)])
def test_recovered_labels_equal_oracle_and_planted_partition(tt, G, b, z):
    H, C, Cp, truth = planted(G, b, z, 8100 + b)
    labels, n = tt.recover_subdomains(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx))
    ref, nref = oracle_recover(Cp.row_ptr, Cp.col_idx)
    got = labels.cpu().numpy()
    assert n == nref and np.array_equal(got, ref)                     # bit-exact against the oracle
    if b < 16:
        return          # 8-row subdomains at z = 0.3 are statistically inseparable (the oracle's groups differ from the planted ones too)
    assert n == G ** 3
    assert np.array_equal(canonical(got), canonical(truth))           # and the generator's partition
    # unpermuted rows: blocks in order
    labels0, n0 = tt.recover_subdomains(C.M, dev(C.row_ptr), dev(C.col_idx))
    assert n0 == G ** 3 and np.array_equal(labels0.cpu().numpy(), np.arange(H.M) // b)


def test_recover_degenerate_inputs(tt):
    # diagonal matrix: singletons
    M = 300
    labels, n = tt.recover_subdomains(M, dev(np.arange(M + 1, dtype=np.int32)), dev(np.arange(M, dtype=np.int32)))
    assert n == M and np.array_equal(labels.cpu().numpy(), np.arange(M))
    # fully dense H (G = 2, z = 0): no recoverable structure, as in the oracle
    H, C, Cp, truth = planted(2, 32, 0.0, 8300)
    assert oracle_recover(Cp.row_ptr, Cp.col_idx) == (None, 0)
    assert tt.recover_subdomains(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx)) == (None, 0)
    # random pattern without structure (symmetrised Bernoulli): whatever the groups are, they equal the oracle's
    rng = np.random.default_rng(5)
    M = 400
    A = rng.random((M, M)) < 0.05
    A = A | A.T | np.eye(M, dtype=bool)
    rp = np.concatenate([[0], np.cumsum(A.sum(1))]).astype(np.int32)
    ci = np.concatenate([np.flatnonzero(A[i]) for i in range(M)]).astype(np.int32)
    ref, nref = oracle_recover(rp, ci)
    labels, n = tt.recover_subdomains(M, dev(rp), dev(ci))
    assert n == nref and np.array_equal(labels.cpu().numpy(), ref)
    # empty rows, rows without a diagonal entry, cliques of different sizes
    rp = np.array([0, 0, 2, 4, 5], np.int32)
    ci = np.array([2, 3, 1, 3, 3], np.int32)
    ref, nref = oracle_recover(rp, ci)
    labels, n = tt.recover_subdomains(4, dev(rp), dev(ci))
    assert n == nref and np.array_equal(labels.cpu().numpy(), ref)
    # errors: workspace / arguments
    import torch
    with pytest.raises(tt.TTDFTError):
        tt.recover_subdomains(-1, dev(rp), dev(ci))


@pytest.mark.parametrize("G,b,z", [(3, 64, 0.3), (3, 128, 0.4)])
def test_unlabelled_permuted_csr_runs_tile_kernels_after_recovery(tt, G, b, z):
    import torch
    H, C, _, (a0, bb) = small_problem(G, b, z, 8200 + b)
    perm = synth.permutation(H.M, 8250 + b)
    Cp = synth.permute_csr(C, perm)
    rp, ci, va = dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values)
    assert tt.h_build_csr(Cp.M, rp, ci, va).info()["kernel"] != 1          # as given: the generic kernel
    Hd = tt.h_build_csr(Cp.M, rp, ci, va, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY, recover=True)
    info = Hd.info()
    assert info["kernel"] == 1 and info["block"] == b and info["reordered"] == 1 and info["nblocks"] == H.nblocks
    N, m = 72, 8
    a, bq, a0q = bounds_for(a0, bb, N, H.M)
    X = synth.dense_normal(H.M, N, 83)
    ref = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, m, a, bq, a0q)
    Y = torch.empty((H.M, N), dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Y, m, a, bq, a0q)
    got = Y.cpu().numpy()
    assert relerr(got, ref) <= 1e-10 and worst_col_relerr(got, ref) <= 1e-9


def test_full_config3_unlabelled_permuted_csr(tt):
    """BASELINE.json config 5 layout (ii) at full size: config 3's H as a symmetrically permuted CSR without labels.  The recovered
    groups are the generator's 1,728 subdomains exactly (integer work: bit-exact), the handle built from them has exactly the
    generator's tiles, and a product in the caller's row order matches the oracle on the permuted CSR."""
    import torch
    cfg = synth.CONFIGS["si"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    nblocks = H.nblocks
    C = synth.bsr_to_csr_nonzeros(H)
    del H
    perm = synth.permutation(cfg.M, cfg.seed + 50)
    Cp = synth.permute_csr(C, perm)
    del C
    rp, ci, va = dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values)
    labels, n = tt.recover_subdomains(cfg.M, rp, ci)
    assert n == cfg.M // cfg.b
    truth = np.empty(cfg.M, np.int32)
    truth[perm] = (np.arange(cfg.M) // cfg.b).astype(np.int32)
    first = np.full(n, cfg.M, np.int64)
    np.minimum.at(first, truth, np.arange(cfg.M))
    assert np.array_equal(np.argsort(np.argsort(first))[truth], labels.cpu().numpy())   # planted groups numbered by smallest row
    Hd = tt.h_build_csr(cfg.M, rp, ci, va, subdomain_of_row=labels)
    info = Hd.info()
    assert info["kernel"] == 1 and info["block"] == cfg.b and info["reordered"] == 1 and info["nblocks"] == nblocks
    del rp, ci, va
    N = 24
    X = synth.dense_normal(cfg.M, N, 8400)
    ref = oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, X)
    Y = torch.empty((cfg.M, N), dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
    got = Y.cpu().numpy()
    assert relerr(got, ref) <= 1e-12 and worst_col_relerr(got, ref) <= 1e-11
