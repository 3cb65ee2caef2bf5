"""A0 reorder (north_star "reorders rows so each localized subdomain's basis functions are
contiguous"): CSR of the symmetrically permuted Hamiltonian P H P^T plus the subdomain index of every row.
The builder must regroup the rows into b x b tiles and every entry point must still take and return X, Y in
the CALLER's (permuted) row order.  Expected values: the CPU oracle on the permuted CSR itself."""
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


def permuted_problem(G, b, z, seed):
    """(H bsr, permuted CSR, labels of the permuted rows, bounds)"""
    H, C, _, (a0, bb) = small_problem(G, b, z, seed)
    perm = synth.permutation(H.M, seed + 50)                 # H'[perm[i], perm[j]] = H[i, j]
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // b).astype(np.int32)    # permuted row perm[i] belongs to subdomain i // b
    return H, Cp, labels, (a0, bb)


def build(t, Cp, labels, flags=0):
    return t.h_build_csr(Cp.M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values), subdomain_of_row=dev(labels), flags=flags)


@pytest.mark.parametrize("G,b,z", [(4, 32, 0.0), (3, 64, 0.3), (2, 96, 0.4), (3, 128, 0.4)])
def test_reordered_build_and_single_steps(tt, G, b, z):
    import torch
    H, Cp, labels, _ = permuted_problem(G, b, z, 3000 + b)
    Hd = build(tt, Cp, labels, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    info = Hd.info()
    assert info["kernel"] == 1 and info["block"] == b and info["reordered"] == 1
    assert info["nblocks"] == H.nblocks                      # the regrouped tiles are exactly the generator's
    N = 70
    X = synth.dense_normal(H.M, N, 81)
    Y0 = synth.dense_normal(H.M, N, 82)
    ref = oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, -0.75, X, 2.5, Y0.copy())
    # without scratch: the generic kernel through the row map
    Y = dev(Y0)
    tt.spmm(Hd, -0.75, dev(X), 2.5, Y)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_SPMM
    # with scratch: gather -> tile kernel (int8 for b >= 64, fp64 tensor cores for b = 32) -> scatter
    for mode in ([tt.MATH_FP64, tt.MATH_I8X7, tt.MATH_I8] if info["i8_planes"] and b >= 64 else [tt.MATH_FP64]):
        Hd.set_math_mode(mode)
        assert tt.step_work_bytes(Hd, N) >= 2 * H.M * N * 8
        Y = dev(Y0)
        tt.spmm(Hd, -0.75, dev(X), 2.5, Y, use_work=True)
        assert relerr(Y.cpu().numpy(), ref) <= TOL_SPMM
        Y = torch.full((H.M, N), float("nan"), dtype=torch.float64, device="cuda")
        tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)      # beta = 0 must not read Y
        assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, X)) <= TOL_SPMM
        alpha, c, beta = 0.173, 9.5, -0.31
        refs = oracle.cheb_step(Cp.row_ptr, Cp.col_idx, Cp.values, alpha, c, beta, X, Y0)
        z = dev(Y0)
        tt.cheb_step(Hd, alpha, c, beta, dev(X), z, z, use_work=True)      # in place over Y_{k-1}
        assert relerr(z.cpu().numpy(), refs) <= TOL_SPMM
    out = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_step(Hd, alpha, c, beta, dev(X), dev(Y0), out)
    assert relerr(out.cpu().numpy(), refs) <= TOL_SPMM


@pytest.mark.parametrize("mode", ["fp64", "i8x7"])
@pytest.mark.parametrize("m,inplace,panel", [(1, False, 0), (1, True, 0), (2, True, 0), (7, False, 48), (7, True, 48), (20, False, 0)])
def test_reordered_filter(tt, mode, m, inplace, panel):
    import torch
    H, Cp, labels, (a0, bb) = permuted_problem(3, 64, 0.3, 3064)
    N = 100
    a, bb, a0 = bounds_for(a0, bb, N, H.M, wide=True)
    Hd = build(tt, Cp, labels)
    Hd.set_math_mode({"fp64": tt.MATH_FP64, "i8x7": tt.MATH_I8X7}[mode])
    X = synth.dense_normal(H.M, N, 91)
    ref = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, m, a, bb, a0)
    Xd = dev(X)
    Yd = Xd if inplace else torch.empty_like(Xd)
    tt.cheb_filter(Hd, Xd, Yd, m, a, bb, a0, panel_cols=panel)
    got = Yd.cpu().numpy()
    assert relerr(got, ref) <= TOL_FILTER
    assert worst_col_relerr(got, ref) <= 10 * TOL_FILTER
    if not inplace:
        assert np.array_equal(Xd.cpu().numpy(), X)


def test_reordered_filter_equals_grouped_filter(tt):
    """Permutation equivariance on the GPU: F_{PHP^T}(PX) = P F_H(X), tile kernels on both
    sides, so the two results agree to rounding of the same arithmetic (bit for bit here: same tiles, same order)."""
    import torch
    H, C, _, (a0, bb) = small_problem(3, 64, 0.3, 3064)
    perm = synth.permutation(H.M, 3064 + 50)
    Cp = synth.permute_csr(C, perm)
    labels = np.empty(H.M, np.int32)
    labels[perm] = (np.arange(H.M) // H.b).astype(np.int32)
    N, m = 64, 9
    a, bb, a0 = bounds_for(a0, bb, N, H.M)
    X = synth.dense_normal(H.M, N, 95)
    Hg = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    Hp = build(tt, Cp, labels)
    Yg = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hg, dev(X), Yg, m, a, bb, a0)
    Yp = torch.empty_like(Yg)
    tt.cheb_filter(Hp, dev(synth.permute_rows(X, perm)), Yp, m, a, bb, a0)
    assert np.array_equal(Yp.cpu().numpy(), synth.permute_rows(Yg.cpu().numpy(), perm))


def test_reordered_host_buffers(tt):
    import torch
    H, Cp, labels, (a0, bb) = permuted_problem(3, 64, 0.3, 3064)
    N, m = 90, 6
    a, bb, a0 = bounds_for(a0, bb, N, H.M)
    Hd = build(tt, Cp, labels)
    X = synth.dense_normal(H.M, N, 97)
    ref = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, m, a, bb, a0)
    Xh = torch.from_numpy(X).pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    tt.cheb_filter_host(Hd, Xh, Yh, m, a, bb, a0, panel_cols=32)
    assert relerr(Yh.numpy(), ref) <= TOL_FILTER


def test_labels_that_do_not_qualify_keep_csr(tt):
    H, Cp, labels, _ = permuted_problem(4, 32, 0.0, 3032)
    bad = labels.copy()
    i = int(np.flatnonzero(bad == 3)[0])
    bad[i] = 4                                    # subdomain 3 owns 31 rows, subdomain 4 owns 33: unequal sizes are padded (to 64)
    Hu = build(tt, Cp, bad)
    assert Hu.info()["kernel"] == 1 and Hu.info()["padded"] == 1 and Hu.info()["block"] == 64
    X = synth.dense_normal(H.M, 20, 86)
    import torch
    Y = torch.empty(H.M, 20, dtype=torch.float64, device="cuda")
    tt.spmm(Hu, 1.0, dev(X), 0.0, Y, use_work=True)
    assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, X)) <= TOL_SPMM
    bad = labels.copy()
    bad[bad == 7] = 9                             # a gap in the labels (no subdomain 7): not the indices 0..nb-1
    assert build(tt, Cp, bad).info()["kernel"] == 0
    bad = labels.copy()
    bad[0] = -1
    assert build(tt, Cp, bad).info()["kernel"] == 0
    bad = labels + 5                              # not the indices 0..nb-1
    assert build(tt, Cp, bad).info()["kernel"] == 0
    assert build(tt, Cp, labels, flags=tt.FORCE_GENERIC).info()["kernel"] == 0


def unequal_problem(G, bmax, lo, z, seed):
    """A planted partition with subdomains of UNEQUAL size: the generator's H (G^3 subdomains of bmax functions) with a random subset
    of every subdomain's functions removed (lo .. bmax kept), then symmetrically permuted.  Returns (permuted CSR, labels, bounds)."""
    H, C, _, (a0, bb) = small_problem(G, bmax, z, seed)
    rng = np.random.default_rng(seed)
    nb = H.M // bmax
    keep = np.zeros(H.M, bool)
    for L in range(nb):
        s = int(rng.integers(lo, bmax + 1))
        keep[L * bmax + rng.choice(bmax, s, replace=False)] = True
    keep[:bmax] = True                                        # one subdomain at full size: the tile size is bmax
    idx = np.nonzero(keep)[0]
    newid = -np.ones(H.M, np.int64)
    newid[idx] = np.arange(len(idx))
    rp = [0]
    ci, va = [], []
    for i in idx:
        cols = C.col_idx[C.row_ptr[i]:C.row_ptr[i + 1]]
        vals = C.values[C.row_ptr[i]:C.row_ptr[i + 1]]
        sel = keep[cols]
        ci.append(newid[cols[sel]])
        va.append(vals[sel])
        rp.append(rp[-1] + int(sel.sum()))
    Cs = synth.CSR(len(idx), np.array(rp, np.int32), np.concatenate(ci).astype(np.int32), np.concatenate(va))
    lab = (idx // bmax).astype(np.int32)
    perm = synth.permutation(Cs.M, seed + 50)
    Cp = synth.permute_csr(Cs, perm)
    labels = np.empty(Cs.M, np.int32)
    labels[perm] = lab
    return Cp, labels, nb, (a0 - 0.5, bb + 0.5)               # deleting rows/columns only shrinks the spectral range (interlacing)


@pytest.mark.parametrize("G,bmax,lo,z", [(3, 128, 80, 0.4), (3, 96, 70, 0.4), (3, 64, 40, 0.3), (4, 32, 20, 0.0)])
def test_unequal_subdomain_sizes_are_padded_to_tiles(tt, G, bmax, lo, z):
    """Labels whose groups differ in size (the Tucker ranks differ per subdomain) still run on the tile kernels: every
    subdomain is padded to the tile size inside h_build, X and Y stay in the caller's row order and size."""
    import torch
    Cp, labels, nb, (a0, bb) = unequal_problem(G, bmax, lo, z, 3300 + bmax)
    M = Cp.M
    assert len(set(np.bincount(labels))) > 3                 # really unequal
    Hd = build(tt, Cp, labels, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    info = Hd.info()
    assert info["kernel"] == 1 and info["block"] == bmax and info["reordered"] == 1 and info["padded"] == 1 and info["M"] == M
    N, m = 70, 9
    a, bq, a0q = bounds_for(a0, bb, N, M)
    X = synth.dense_normal(M, N, 83)
    Y0 = synth.dense_normal(M, N, 84)
    ref_mm = oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, -0.75, X, 2.5, Y0.copy())
    ref_f = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, m, a, bq, a0q)
    Y = dev(Y0)
    tt.spmm(Hd, -0.75, dev(X), 2.5, Y)                        # without scratch: the generic kernel through the row map
    assert relerr(Y.cpu().numpy(), ref_mm) <= TOL_SPMM
    modes = [tt.MATH_FP64] + ([tt.MATH_I8X7, tt.MATH_I8] if info["i8_planes"] and bmax >= 64 else [])
    for mode in modes:
        Hd.set_math_mode(mode)
        Y = dev(Y0)
        tt.spmm(Hd, -0.75, dev(X), 2.5, Y, use_work=True)     # gather -> tile kernel on the padded space -> scatter
        assert relerr(Y.cpu().numpy(), ref_mm) <= TOL_SPMM
        for inplace in (False, True):
            Xd = dev(X)
            Yd = Xd if inplace else torch.full((M, N), float("nan"), dtype=torch.float64, device="cuda")
            tt.cheb_filter(Hd, Xd, Yd, m, a, bq, a0q, panel_cols=48)
            got = Yd.cpu().numpy()
            assert relerr(got, ref_f) <= TOL_FILTER and worst_col_relerr(got, ref_f) <= 10 * TOL_FILTER
        Yd = torch.empty((M, N), dtype=torch.float64, device="cuda")
        tt.cheb_filter(Hd, dev(X), Yd, 4, a, bq, a0q)          # even degree, one panel
        assert relerr(Yd.cpu().numpy(), oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, X, 4, a, bq, a0q)) <= TOL_FILTER
    # Lanczos bounds and the projection on the padded handle
    v0 = synth.dense_normal(M, 1, 85).reshape(-1)
    la0, lb, _ = tt.lanczos_bounds(Hd, dev(v0), 20)
    ra0, rb, _ = oracle.lanczos_bounds(Cp.row_ptr, Cp.col_idx, Cp.values, v0, 20)
    assert abs(la0 - ra0) <= 1e-9 * (rb - ra0) and abs(lb - rb) <= 1e-9 * (rb - ra0)
    Hd.set_math_mode(tt.MATH_AUTO)
    G_ = torch.empty((N, N), dtype=torch.float64, device="cuda")
    tt.project(Hd, dev(X), G_)
    assert relerr(G_.cpu().numpy(), oracle.project(Cp.row_ptr, Cp.col_idx, Cp.values, X)) <= 1e-12
    # too much padding (tiny groups): the generic format is kept
    tiny = (np.arange(M) // 3).astype(np.int32)
    Hg = tt.h_build_csr(M, dev(Cp.row_ptr), dev(Cp.col_idx), dev(Cp.values), subdomain_of_row=dev(tiny))
    assert Hg.info()["kernel"] == 0 and Hg.info()["padded"] == 0
