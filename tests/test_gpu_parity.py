"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are north_star's: relative Frobenius error <= 1e-12 per SpMM / single
fused step and <= 1e-10 after a degree-m filter, normalised by ||Y||_F."""
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


def build_bsr(t, H, flags=0):
    return t.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=flags)


def build_csr(t, C, labels=None, flags=0):
    return t.h_build_csr(C.M, dev(C.row_ptr), dev(C.col_idx), dev(C.values),
                         subdomain_of_row=None if labels is None else dev(labels), flags=flags)


# ---------------------------------------------------------------- config 1 (tiny), all entry points
@pytest.mark.parametrize("N,ld", [(32, 32), (33, 40), (1, 2), (130, 130), (257, 300)])
def test_spmm_tiny_bsr(tt, N, ld):
    import torch
    H, C, (rp, col, val), _ = small_problem(4, 32, 0.0, 1001)
    Hd = build_bsr(tt, H, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    assert Hd.info()["kernel"] == 1
    X = synth.dense_normal(H.M, N, 11)
    Y0 = synth.dense_normal(H.M, N, 12)
    Xd = torch.zeros(H.M, ld, dtype=torch.float64, device="cuda")
    Xd[:, :N] = dev(X)
    Yd = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, Xd[:, :N], 0.0, Yd[:, :N])          # beta = 0 must not read Y
    ref = oracle.spmm(rp, col, val, 1.0, X)
    got = Yd[:, :N].cpu().numpy()
    assert relerr(got, ref) <= TOL_SPMM
    assert worst_col_relerr(got, ref) <= 10 * TOL_SPMM
    if ld > N:
        assert torch.isnan(Yd[:, N:]).all()              # nothing written outside the view
    Yd[:, :N] = dev(Y0)
    tt.spmm(Hd, -0.75, Xd[:, :N], 2.5, Yd[:, :N])
    ref = oracle.spmm(rp, col, val, -0.75, X, 2.5, Y0.copy())
    assert relerr(Yd[:, :N].cpu().numpy(), ref) <= TOL_SPMM
    # alpha = 0: H and X are not read
    Yd[:, :N] = dev(Y0)
    tt.spmm(Hd, 0.0, torch.full_like(Xd, float("nan"))[:, :N], 2.0, Yd[:, :N])
    assert relerr(Yd[:, :N].cpu().numpy(), 2.0 * Y0) <= 1e-15


@pytest.mark.parametrize("N", [32, 50])
def test_cheb_step_tiny(tt, N):
    import torch
    H, C, (rp, col, val), _ = small_problem(4, 32, 0.0, 1001)
    Hd = build_bsr(tt, H)
    Yk = synth.dense_normal(H.M, N, 21)
    Ykm1 = synth.dense_normal(H.M, N, 22)
    al, c, be = -0.21, 10.3, -0.17
    ref = oracle.cheb_step(rp, col, val, al, c, be, Yk, Ykm1)
    out = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_step(Hd, al, c, be, dev(Yk), dev(Ykm1), out)
    assert relerr(out.cpu().numpy(), ref) <= TOL_SPMM
    # in place over Ykm1
    z = dev(Ykm1)
    tt.cheb_step(Hd, al, c, be, dev(Yk), z, z)
    assert relerr(z.cpu().numpy(), ref) <= TOL_SPMM
    # first step: beta term absent
    ref1 = oracle.cheb_step(rp, col, val, al, c, 0.0, Yk, None)
    tt.cheb_step(Hd, al, c, 123.0, dev(Yk), None, out)
    assert relerr(out.cpu().numpy(), ref1) <= TOL_SPMM


def test_cheb_scalars_match_paper_recurrence(tt):
    from fractions import Fraction
    c, al, be = tt.cheb_scalars(5, 2.0, 10.0, 0.0)
    e, cc = Fraction(4), Fraction(6)
    sig = e / (0 - cc)
    gamma = 2 / sig
    assert c == 6.0 and al[0] == pytest.approx(float(sig / e), rel=1e-15) and be[0] == 0.0
    for k in range(1, 5):
        s2 = 1 / (gamma - sig)
        assert al[k] == pytest.approx(float(2 * s2 / e), rel=1e-15)
        assert be[k] == pytest.approx(float(-sig * s2), rel=1e-15)
        sig = s2


@pytest.mark.parametrize("m", [0, 1, 2, 3, 10, 11])
@pytest.mark.parametrize("inplace", [False, True])
def test_filter_tiny_full(tt, m, inplace):
    import torch
    cfg = synth.CONFIGS["tiny"]
    H, C, (rp, col, val), (a0, b) = small_problem(cfg.G, cfg.b, cfg.z, cfg.seed)
    a, b, a0 = bounds_for(a0, b, cfg.N, H.M)
    Hd = build_bsr(tt, H)
    X = synth.dense_normal(H.M, cfg.N, cfg.seed)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, b, a0)
    Xd = dev(X)
    Yd = Xd if inplace else torch.empty_like(Xd)
    tt.cheb_filter(Hd, Xd, Yd, m, a, b, a0)
    got = Yd.cpu().numpy()
    assert relerr(got, ref) <= TOL_FILTER
    assert worst_col_relerr(got, ref) <= 10 * TOL_FILTER
    if not inplace:
        assert np.array_equal(Xd.cpu().numpy(), X)       # input untouched


@pytest.mark.parametrize("N,panel", [(100, 48), (100, 100), (70, 32), (33, 16), (37, 7)])
def test_filter_panels_and_ragged(tt, N, panel):
    """Panel width not dividing N, ragged N, odd panel width (misaligned views -> generic kernel)."""
    import torch
    H, C, (rp, col, val), (a0, b) = small_problem(4, 32, 0.0, 1001)
    a, b, a0 = bounds_for(a0, b, 32, H.M, wide=True)       # wide gap: T_7(t0) large dynamic range
    Hd = build_bsr(tt, H)
    X = synth.dense_normal(H.M, N, 31)
    ref = oracle.cheb_filter(rp, col, val, X, 7, a, b, a0)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Y, 7, a, b, a0, panel_cols=panel)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_FILTER
    assert worst_col_relerr(Y.cpu().numpy(), ref) <= 10 * TOL_FILTER


def test_filter_host_buffers(tt):
    import torch
    H, C, (rp, col, val), (a0, b) = small_problem(4, 32, 0.0, 1001)
    a, b, a0 = bounds_for(a0, b, 32, H.M)
    Hd = build_bsr(tt, H)
    N = 200
    X = synth.dense_normal(H.M, N, 41)
    ref = oracle.cheb_filter(rp, col, val, X, 10, a, b, a0)
    Xh = torch.from_numpy(X).pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    tt.cheb_filter_host(Hd, Xh, Yh, 10, a, b, a0, panel_cols=64)   # 4 panels, double buffered
    assert relerr(Yh.numpy(), ref) <= TOL_FILTER


@pytest.mark.parametrize("G,b,N,mode", [(4, 32, 700, "FP64"), (3, 64, 2500, "I8X7"), (3, 64, 200, "I8X7")])
def test_filter_host_default_panel_schedule(tt, G, b, N, mode):
    """panel_cols = 0 on host buffers: a ramp of panel widths, narrow first and last (N = 700: 128 | 444 | 128,
    N = 2,500: 256 | 768 | 452 | 768 | 256, N = 200: one panel).  Every column equals the device-resident filter's bit for bit (the
    result of a column does not depend on the panels), and sampled columns the oracle's."""
    import torch
    H, C, _, (a0, bb) = small_problem(G, b, 0.3, 1300 + b)
    a, bb, a0 = bounds_for(a0, bb, 64, H.M)
    Hd = build_bsr(tt, H)
    Hd.set_math_mode(getattr(tt, "MATH_" + mode))
    X = synth.dense_normal(H.M, N, 43)
    Xh = torch.from_numpy(X).pin_memory()
    Yh = torch.full((H.M, N), float("nan"), dtype=torch.float64).pin_memory()
    tt.cheb_filter_host(Hd, Xh, Yh, 9, a, bb, a0, panel_cols=0)
    Yd = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Yd, 9, a, bb, a0)
    assert torch.equal(Yh, Yd.cpu())
    cols = sorted({0, 63, 64, 127, 128, 255, 256, N // 2, N - 129, N - 128, N - 1} & set(range(N)))
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, np.ascontiguousarray(X[:, cols]), 9, a, bb, a0)
    assert worst_col_relerr(Yh.numpy()[:, cols], ref) <= TOL_FILTER


# ---------------------------------------------------------------- other tile sizes (several tiles + ragged tail)
@pytest.mark.parametrize("G,b,z,N", [(3, 64, 0.3, 200), (2, 96, 0.4, 130), (3, 128, 0.4, 300)])
def test_filter_other_block_sizes(tt, G, b, z, N):
    import torch
    H, C, (rp, col, val), (a0, bb) = small_problem(G, b, z, 2000 + b)
    a, bb, a0 = bounds_for(a0, bb, N, H.M)
    Hd = build_bsr(tt, H)
    assert Hd.info()["kernel"] == 1 and Hd.info()["block"] == b
    X = synth.dense_normal(H.M, N, 51)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(rp, col, val, 1.0, X)) <= TOL_SPMM
    m = 20
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, bb, a0)   # oracle on the non-zeros only
    tt.cheb_filter(Hd, dev(X), Y, m, a, bb, a0, panel_cols=128)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_FILTER
    assert worst_col_relerr(Y.cpu().numpy(), ref) <= 10 * TOL_FILTER


# ---------------------------------------------------------------- CSR inputs
def test_csr_generic_and_permuted(tt):
    import torch
    H, C, _, (a0, b) = small_problem(4, 32, 0.0, 1001)
    N = 40
    a, b, a0 = bounds_for(a0, b, 32, H.M)
    X = synth.dense_normal(H.M, N, 61)
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, 10, a, b, a0)
    Hc = build_csr(tt, C, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    assert Hc.info()["kernel"] == 0
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hc, dev(X), Y, 10, a, b, a0)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_FILTER
    # symmetric random permutation (BASELINE.json config 5's irregular layout): F_{PHP^T}(PX) = P F_H(X)
    perm = synth.permutation(H.M, 5)
    Cp = synth.permute_csr(C, perm)
    Hp = build_csr(tt, Cp, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)
    Xp = synth.permute_rows(X, perm)
    tt.cheb_filter(Hp, dev(Xp), Y, 10, a, b, a0)
    refp = oracle.cheb_filter(Cp.row_ptr, Cp.col_idx, Cp.values, Xp, 10, a, b, a0)
    assert relerr(Y.cpu().numpy(), refp) <= TOL_FILTER
    assert relerr(Y.cpu().numpy(), synth.permute_rows(ref, perm)) <= TOL_FILTER
    tt.spmm(Hp, 1.0, dev(Xp), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 1.0, Xp)) <= TOL_SPMM


@pytest.mark.parametrize("N,ld", [(1, 1), (7, 9), (16, 16), (31, 40), (32, 32), (33, 34), (50, 64), (64, 64)])
def test_csr_narrow_panels(tt, N, ld):
    """Panels of <= 64 columns on a CSR run K2's narrow variants (four / two entries of a row per warp step): every width, padded leading
    dimensions, the fused step with all three terms, rows whose length is not a multiple of 4 or 32 (z = 0.5), an empty row."""
    import torch
    H, C, _, _ = small_problem(3, 32, 0.5, 1007)
    perm = synth.permutation(H.M, 9)
    Cp = synth.permute_csr(C, perm)
    Hp = build_csr(tt, Cp)
    assert Hp.info()["kernel"] == 0
    X = synth.dense_normal(H.M, N, 63)
    Z = synth.dense_normal(H.M, N, 64)
    Xd = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
    Zd = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
    Od = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
    Xd[:, :N] = dev(X)
    Zd[:, :N] = dev(Z)
    tt.cheb_step(Hp, 0.7, -1.3, -0.4, Xd[:, :N], Zd[:, :N], Od[:, :N])
    ref = oracle.cheb_step(Cp.row_ptr, Cp.col_idx, Cp.values, 0.7, -1.3, -0.4, X, Z)
    assert relerr(Od[:, :N].cpu().numpy(), ref) <= TOL_SPMM
    assert bool(torch.isnan(Od[:, N:]).all())                     # nothing written outside the view
    Y = dev(Z)
    tt.spmm(Hp, 2.0, dev(X), 0.5, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(Cp.row_ptr, Cp.col_idx, Cp.values, 2.0, X, 0.5, Z.copy())) <= TOL_SPMM
    # a matrix with an empty row: row 5 and column 5 removed
    keep = (np.repeat(np.arange(Cp.M), np.diff(Cp.row_ptr)) != 5) & (Cp.col_idx != 5)
    rp = np.zeros(Cp.M + 1, np.int64)
    np.add.at(rp, np.repeat(np.arange(Cp.M), np.diff(Cp.row_ptr))[keep] + 1, 1)
    E = synth.CSR(Cp.M, np.cumsum(rp).astype(np.int32), Cp.col_idx[keep].copy(), Cp.values[keep].copy())
    He = build_csr(tt, E)
    Y = dev(Z)
    tt.spmm(He, 1.0, dev(X), -1.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(E.row_ptr, E.col_idx, E.values, 1.0, X, -1.0, Z.copy())) <= TOL_SPMM


def test_csr_with_subdomain_hint_builds_tiles(tt):
    import torch
    H, C, (rp, col, val), (a0, b) = small_problem(4, 32, 0.0, 1001)
    labels = (np.arange(H.M) // H.b).astype(np.int32) * 3 + 7      # non-decreasing, equal groups of 32
    Hh = build_csr(tt, C, labels=labels)
    info = Hh.info()
    assert info["kernel"] == 1 and info["block"] == 32 and info["nblocks"] == H.nblocks
    N = 64
    X = synth.dense_normal(H.M, N, 71)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hh, 1.0, dev(X), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, X)) <= TOL_SPMM
    # labels that are not grouped -> CSR is kept
    bad = labels.copy()
    bad[5] = 999999
    assert build_csr(tt, C, labels=bad).info()["kernel"] == 0


def test_generic_kernel_on_bsr(tt):
    import torch
    H, C, (rp, col, val), _ = small_problem(4, 32, 0.0, 1001)
    Hg = build_bsr(tt, H, flags=tt.FORCE_GENERIC)
    assert Hg.info()["kernel"] == 0
    X = synth.dense_normal(H.M, 19, 81)
    Y = torch.empty(H.M, 19, dtype=torch.float64, device="cuda")
    tt.spmm(Hg, 1.0, dev(X), 0.0, Y)
    assert relerr(Y.cpu().numpy(), oracle.spmm(rp, col, val, 1.0, X)) <= TOL_SPMM


# ---------------------------------------------------------------- degenerate inputs and errors
def test_degenerate_and_errors(tt):
    import torch
    H, C, _, (a0, b) = small_problem(4, 32, 0.0, 1001)
    Hd = build_bsr(tt, H)
    X = dev(synth.dense_normal(H.M, 8, 1))
    Y = torch.zeros_like(X)
    with pytest.raises(tt.TTDFTError) as e:
        tt.cheb_filter(Hd, X, Y, -1, 1.0, 2.0, 0.0)
    assert e.value.status_name == "INVALID_ARG"
    with pytest.raises(tt.TTDFTError):
        tt.cheb_filter(Hd, X, Y, 3, 2.0, 1.0, 0.0)          # a > b
    with pytest.raises(tt.TTDFTError):
        tt.spmm(Hd, 1.0, X, 0.0, X)                          # X aliases Y
    with pytest.raises(tt.TTDFTError):
        tt.cheb_filter(Hd, X, Y, 4, 1.0, 2.0, 0.0, work=torch.empty(64, dtype=torch.uint8, device="cuda"))
    assert torch.count_nonzero(Y) == 0                       # outputs untouched on error
    # not symmetric / unsorted inputs are reported on request
    vals = H.values.copy()
    vals[1, 0, 1] += 1.0
    with pytest.raises(tt.TTDFTError) as e:
        tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(vals), flags=tt.CHECK_SYMMETRY | tt.CHECK_SORTED)
    assert e.value.status_name == "NOT_SYMMETRIC"
    cols = C.col_idx.copy()
    cols[[0, 1]] = cols[[1, 0]]
    with pytest.raises(tt.TTDFTError) as e:
        tt.h_build_csr(C.M, dev(C.row_ptr), dev(cols), dev(C.values), flags=tt.CHECK_SORTED)
    assert e.value.status_name == "INVALID_ARG"
    # empty block rows and a 1-block matrix
    rp = np.array([0, 1, 1], np.int32)
    Hs = tt.h_build_bsr(64, 32, dev(rp), dev(np.array([0], np.int32)), dev(np.eye(32).reshape(1, 32, 32) * 2.0))
    X2 = dev(synth.dense_normal(64, 5, 2))
    Y2 = torch.empty_like(X2)
    tt.spmm(Hs, 1.0, X2, 0.0, Y2)
    ref = X2.cpu().numpy() * 2.0
    ref[32:] = 0.0
    assert np.array_equal(Y2.cpu().numpy(), ref)


def test_launch_counter_and_probe(tt):
    n0 = tt.launch_count()
    H, C, _, _ = small_problem(4, 32, 0.0, 1001)
    Hd = build_bsr(tt, H)
    X = dev(synth.dense_normal(H.M, 8, 1))
    import torch
    Y = torch.empty_like(X)
    n1 = tt.launch_count()
    assert n1 == n0 + 2                      # the builder's two digit-plane kernels (row scales, planes)
    tt.spmm(Hd, 1.0, X, 0.0, Y)
    assert tt.launch_count() == n1 + 1       # one fused kernel per product
    tt.timing_enable(True)
    tt.spmm(Hd, 1.0, X, 0.0, Y)
    tt.timing_enable(False)
    ms, n = tt.timing_read("bsr_dmma")
    assert n == 1 and ms > 0.0
    assert tt.timing_read("bsr_dmma") == (0.0, 0)
    assert tt.probe_fp64_peak(1, 50) > 5.0
