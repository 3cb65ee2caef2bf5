"""Packed tile storage (bsr_packed.cuh; SURVEY.md 7 "Small-N regime", 8(f)-4 storage variants): a handle built
with TTDFT_PACKED streams bit maps + non-zero values instead of dense tiles for ncols <= 16.  The decoded operand is the dense tile bit for bit and
the tensor-core loop is kernel K1's own, so the result must equal the dense path's EXACTLY and the oracle's within 1e-12."""
import numpy as np
import pytest

import oracle
import synth
from util import relerr, small_problem

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


@pytest.mark.parametrize("G,b,z", [(4, 32, 0.0), (3, 64, 0.3), (3, 96, 0.4), (3, 128, 0.4), (2, 128, 0.9)])
@pytest.mark.parametrize("N,ld", [(1, 2), (7, 7), (16, 16), (12, 20)])
def test_packed_products_equal_dense_and_oracle(tt, G, b, z, N, ld):
    import torch
    H, C, _, _ = small_problem(G, b, z, 9500 + b)
    Hp = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY | tt.PACKED)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    ip, idn = Hp.info(), Hd.info()
    nnz = int(np.count_nonzero(H.values))
    assert idn["packed_bytes"] == 0
    # non-zeros (8 B each, every 16-column slab padded to an even count) + 4 B of header per tile row and slab
    nslabs = H.nblocks * (b // 16)
    assert 8 * nnz + 4 * b * nslabs <= ip["packed_bytes"] <= 8 * (nnz + nslabs) + 4 * b * nslabs
    assert ip["storage_bytes"] > idn["storage_bytes"]
    X = synth.dense_normal(H.M, N, 201)
    Z = synth.dense_normal(H.M, N, 202)
    Xd = torch.zeros(H.M, ld, dtype=torch.float64, device="cuda")
    Xd[:, :N] = dev(X)
    alpha, c, beta = 0.173, 9.5, -0.31
    ref_mm = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, X)
    ref_st = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, alpha, c, beta, X, Z)
    outs = []
    for Hh in (Hp, Hd):
        Y = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
        tt.spmm(Hh, 1.0, Xd[:, :N], 0.0, Y[:, :N])
        O = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
        tt.cheb_step(Hh, alpha, c, beta, Xd[:, :N], dev(Z), O[:, :N])
        if ld > N:
            assert torch.isnan(Y[:, N:]).all() and torch.isnan(O[:, N:]).all()
        outs.append((Y[:, :N].cpu().numpy(), O[:, :N].cpu().numpy()))
        assert relerr(outs[-1][0], ref_mm) <= 1e-12 and relerr(outs[-1][1], ref_st) <= 1e-12
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    # in place over Y_{k-1}, and the filter of a narrow block in fp64 mode (every step streams the packed tiles)
    zz = dev(Z)
    tt.cheb_step(Hp, alpha, c, beta, Xd[:, :N], zz, zz)
    assert np.array_equal(zz.cpu().numpy(), outs[0][1])


def test_packed_from_labelled_csr_and_lanczos(tt):
    """The packed copy is also built when the tiles come from a CSR regrouped by subdomain labels, and the one-column products
    of ttdft_lanczos_bounds run on it (same bounds as the oracle's Lanczos)."""
    import torch
    H, C, _, _ = small_problem(3, 64, 0.3, 9600)
    perm = synth.permutation(H.M, 9650)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // H.b).astype(np.int32)
    Hd = tt.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values), subdomain_of_row=dev(labels), flags=tt.PACKED)
    inf = Hd.info()
    assert inf["reordered"] == 1 and inf["packed_bytes"] > 8 * C.nnz
    v0 = synth.dense_normal(H.M, 1, 9600, synth.STREAM_V0).reshape(-1)
    a0, b, theta = tt.lanczos_bounds(Hd, dev(v0), 20)
    ra0, rb, _ = oracle.lanczos_bounds(Cp.row_ptr, Cp.col_idx, Cp.values, v0, 20)
    assert abs(a0 - ra0) <= 1e-9 * (rb - ra0) and abs(b - rb) <= 1e-9 * (rb - ra0)
    Hb = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=tt.PACKED)
    X = synth.dense_normal(H.M, 9, 203)
    Y = torch.empty(H.M, 9, dtype=torch.float64, device="cuda")
    tt.spmm(Hb, 2.0, dev(X), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(C.row_ptr, C.col_idx, C.values, 2.0, X)) <= 1e-12
