"""GPU parity of the int8 digit-plane path (kernel K3, TTDFT_MATH_I8 / TTDFT_MATH_I8X7) against the
CPU oracle.

Same tolerances as the fp64 path (north_star): <= 1e-12 relative Frobenius per SpMM / fused step,
<= 1e-10 after a filter.  K3 splits every operand exactly into 6 (I8) or 7 (I8X7) balanced base-256
digits below its row / column maximum and accumulates in exact integers, so
the measured error is expected around 1e-14 (47 bits) and 1e-16..1e-15 (55 bits: the fp64 rounding
of the epilogue dominates); ACC_SPMM pins that, so that a lost digit plane or level fails."""
import numpy as np
import pytest

import oracle
import synth
from util import bounds_for, relerr, small_problem, worst_col_relerr

pytestmark = pytest.mark.gpu

TOL_SPMM = 1e-12
TOL_FILTER = 1e-10
ACC = {"i8": 2e-13,    # what 47-bit operands must deliver on these inputs
       "i8x7": 4e-15}  # 55-bit operands: as accurate as an fp64 dot product
ACC_SPMM = ACC["i8"]


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2110_15853_b200 as t
    assert torch.cuda.is_available()
    return t


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def build_i8(t, H, flags=0, mode="i8"):
    Hd = t.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=flags)
    assert Hd.info()["i8_planes"] == 7
    want = {"i8": t.MATH_I8, "i8x7": t.MATH_I8X7}[mode]
    Hd.set_math_mode(want)
    assert Hd.info()["math"] == want
    return Hd


@pytest.mark.parametrize("mode", ["i8", "i8x7"])
@pytest.mark.parametrize("N,ld", [(32, 32), (33, 40), (1, 2), (64, 64), (130, 130), (257, 300)])
def test_spmm_ws_tiny(tt, N, ld, mode):
    import torch
    ACC_SPMM = ACC[mode]
    H, C, (rp, col, val), _ = small_problem(4, 32, 0.0, 1001)
    Hd = build_i8(tt, H, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY, mode=mode)
    assert tt.step_work_bytes(Hd, N) > 0
    X = synth.dense_normal(H.M, N, 11)
    Y0 = synth.dense_normal(H.M, N, 12)
    Xd = torch.zeros(H.M, ld, dtype=torch.float64, device="cuda")
    Xd[:, :N] = dev(X)
    Yd = torch.full((H.M, ld), float("nan"), dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, Xd[:, :N], 0.0, Yd[:, :N], use_work=True)      # beta = 0 must not read Y
    ref = oracle.spmm(rp, col, val, 1.0, X)
    got = Yd[:, :N].cpu().numpy()
    assert relerr(got, ref) <= ACC_SPMM
    assert worst_col_relerr(got, ref) <= 10 * ACC_SPMM
    if ld > N:
        assert torch.isnan(Yd[:, N:]).all()                           # nothing written outside the view
    Yd[:, :N] = dev(Y0)
    tt.spmm(Hd, -0.75, Xd[:, :N], 2.5, Yd[:, :N], use_work=True)
    ref = oracle.spmm(rp, col, val, -0.75, X, 2.5, Y0.copy())
    assert relerr(Yd[:, :N].cpu().numpy(), ref) <= TOL_SPMM


@pytest.mark.parametrize("N", [32, 50])
def test_cheb_step_ws_tiny(tt, N):
    import torch
    H, C, (rp, col, val), _ = small_problem(4, 32, 0.0, 1001)
    Hd = build_i8(tt, H)
    Yk = synth.dense_normal(H.M, N, 21)
    Ykm1 = synth.dense_normal(H.M, N, 22)
    alpha, c, beta = 0.173, 9.5, -0.31
    ref = oracle.cheb_step(rp, col, val, alpha, c, beta, Yk, Ykm1)
    out = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_step(Hd, alpha, c, beta, dev(Yk), dev(Ykm1), out, use_work=True)
    assert relerr(out.cpu().numpy(), ref) <= TOL_SPMM
    # in place over Y_{k-1}
    z = dev(Ykm1)
    tt.cheb_step(Hd, alpha, c, beta, dev(Yk), z, z, use_work=True)
    assert relerr(z.cpu().numpy(), ref) <= TOL_SPMM
    # first step: no beta term
    ref1 = oracle.cheb_step(rp, col, val, alpha, c, 0.0, Yk, None)
    tt.cheb_step(Hd, alpha, c, 123.0, dev(Yk), None, out, use_work=True)
    assert relerr(out.cpu().numpy(), ref1) <= TOL_SPMM


@pytest.mark.parametrize("mode", ["i8", "i8x7"])
@pytest.mark.parametrize("m", [1, 2, 3, 10, 11])
@pytest.mark.parametrize("inplace", [False, True])
def test_filter_tiny_full_i8(tt, m, inplace, mode):
    import torch
    cfg = synth.CONFIGS["tiny"]
    H, C, (rp, col, val), (a0, b) = small_problem(cfg.G, cfg.b, cfg.z, cfg.seed)
    a, b, a0 = bounds_for(a0, b, cfg.N, H.M)
    Hd = build_i8(tt, H, mode=mode)
    X = synth.dense_normal(H.M, cfg.N, cfg.seed)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, b, a0)
    Xd = dev(X)
    Yd = Xd if inplace else torch.empty_like(Xd)
    tt.cheb_filter(Hd, Xd, Yd, m, a, b, a0)
    got = Yd.cpu().numpy()
    assert relerr(got, ref) <= TOL_FILTER
    assert worst_col_relerr(got, ref) <= 10 * TOL_FILTER
    if not inplace:
        assert np.array_equal(Xd.cpu().numpy(), X)


@pytest.mark.parametrize("N,panel", [(100, 48), (100, 100), (70, 32), (33, 16), (37, 7)])
def test_filter_panels_and_ragged_i8(tt, N, panel):
    """Panel width not dividing N, ragged N, odd panel width (unaligned views -> scalar epilogue)."""
    import torch
    H, C, (rp, col, val), (a0, b) = small_problem(4, 32, 0.0, 1001)
    a, b, a0 = bounds_for(a0, b, 32, H.M, wide=True)
    Hd = build_i8(tt, H)
    X = synth.dense_normal(H.M, N, 31)
    ref = oracle.cheb_filter(rp, col, val, X, 7, a, b, a0)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Y, 7, a, b, a0, panel_cols=panel)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_FILTER
    assert worst_col_relerr(Y.cpu().numpy(), ref) <= 10 * TOL_FILTER


@pytest.mark.parametrize("mode", ["i8", "i8x7"])
@pytest.mark.parametrize("G,b,z,N", [(3, 64, 0.3, 200), (2, 96, 0.4, 130), (3, 128, 0.4, 300)])
def test_other_block_sizes_i8(tt, G, b, z, N, mode):
    import torch
    ACC_SPMM = ACC[mode]
    H, C, (rp, col, val), (a0, bb) = small_problem(G, b, z, 2000 + b)
    a, bb, a0 = bounds_for(a0, bb, N, H.M)
    Hd = build_i8(tt, H, mode=mode)
    X = synth.dense_normal(H.M, N, 51)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
    assert relerr(Y.cpu().numpy(), oracle.spmm(rp, col, val, 1.0, X)) <= ACC_SPMM
    m = 20
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, bb, a0)
    tt.cheb_filter(Hd, dev(X), Y, m, a, bb, a0, panel_cols=128)
    assert relerr(Y.cpu().numpy(), ref) <= TOL_FILTER
    assert worst_col_relerr(Y.cpu().numpy(), ref) <= 10 * TOL_FILTER
    # the fp64 tensor-core path on the same handle agrees with the same oracle
    Hd.set_math_mode(tt.MATH_FP64)
    Y2 = torch.empty_like(Y)
    tt.cheb_filter(Hd, dev(X), Y2, m, a, bb, a0, panel_cols=128)
    assert relerr(Y2.cpu().numpy(), ref) <= TOL_FILTER


def test_column_dynamic_range_and_zero_columns(tt):
    """Per-column scaling: columns 60 orders of magnitude apart, an all-zero column, a column with one
    huge entry -- every column keeps its own relative accuracy."""
    import torch
    H, C, (rp, col, val), _ = small_problem(3, 64, 0.3, 2064)
    Hd = build_i8(tt, H)
    N = 70
    X = synth.dense_normal(H.M, N, 61)
    scale = 10.0 ** np.linspace(-30, 30, N)
    X = X * scale[None, :]
    X[:, 5] = 0.0
    X[7, 9] = 1e6 * np.abs(X[:, 9]).max()          # one dominant entry: the rest of the column loses bits
    ref = oracle.spmm(rp, col, val, 1.0, X)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
    got = Y.cpu().numpy()
    assert np.all(got[:, 5] == 0.0)
    cols = [j for j in range(N) if j not in (5, 9)]
    assert worst_col_relerr(got[:, cols], ref[:, cols]) <= 10 * ACC_SPMM
    assert worst_col_relerr(got[:, [9]], ref[:, [9]]) <= TOL_SPMM    # still norm-wise accurate


def test_no_i8_flag_and_mode_errors(tt):
    H, C, _, _ = small_problem(4, 32, 0.0, 1001)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values), flags=tt.NO_I8)
    assert Hd.info()["i8_planes"] == 0 and Hd.info()["math"] == tt.MATH_FP64
    with pytest.raises(tt.TTDFTError) as e:
        Hd.set_math_mode(tt.MATH_I8)
    assert e.value.status_name == "UNSUPPORTED"
    with pytest.raises(tt.TTDFTError):
        Hd.set_math_mode(tt.MATH_I8X7)
    with pytest.raises(tt.TTDFTError):
        Hd.set_math_mode(7)
    assert tt.step_work_bytes(Hd, 64) == 0


def test_auto_mode_is_i8x7_for_wide_tiles(tt):
    """TTDFT_MATH_AUTO: 7 planes for tile size >= 64, fp64 DMMA below; work sizes follow the mode."""
    H, C, _, _ = small_problem(3, 64, 0.3, 2064)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    assert Hd.info()["math"] == tt.MATH_I8X7
    w7 = tt.step_work_bytes(Hd, 64)
    Hd.set_math_mode(tt.MATH_I8)
    w6 = tt.step_work_bytes(Hd, 64)
    assert w7 > w6 > 0
    H, C, _, _ = small_problem(4, 32, 0.0, 1001)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    assert Hd.info()["math"] == tt.MATH_FP64


@pytest.mark.parametrize("cluster,hints", [("1", "1"), ("2", "0"), ("2", "2"), ("4", "1"), ("8", "1")])
def test_cluster_sizes_and_l2_hints(tt, cluster, hints):
    """Every cluster size of K3 (TMA multicast of the H planes across 1/2/4/8 CTAs, incl. the single-CTA remainder launch
    when the tile count is not a multiple of the cluster size) and every L2-hint mode gives the same bits."""
    import os
    import torch
    H, C, (rp, col, val), (a0, bb) = small_problem(3, 128, 0.4, 2128)
    N, m = 5 * 64 + 7, 5                                     # 6 column tiles: 4 + remainder 2 under 4-CTA clusters
    a, bb, a0 = bounds_for(a0, bb, N, H.M, wide=True)
    X = synth.dense_normal(H.M, N, 71)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)
    out = {}
    for env in (None, (cluster, hints)):
        for k in ("TTDFT_K3_CLUSTER", "TTDFT_K3_L2HINTS"):
            os.environ.pop(k, None)
        if env:
            os.environ["TTDFT_K3_CLUSTER"], os.environ["TTDFT_K3_L2HINTS"] = env
        try:
            Hd = build_i8(tt, H, mode="i8x7")
            Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
            tt.cheb_filter(Hd, dev(X), Y, m, a, bb, a0)
            out[env] = Y.cpu().numpy()
        finally:
            for k in ("TTDFT_K3_CLUSTER", "TTDFT_K3_L2HINTS"):
                os.environ.pop(k, None)
    assert relerr(out[None], ref) <= TOL_FILTER
    assert np.array_equal(out[None], out[(cluster, hints)])


def test_row_dynamic_range_and_zero_rows(tt):
    """Per-row scaling of H: rows 40 orders of magnitude apart, an all-zero row, a row with only its diagonal entry -- every row
    keeps its own relative accuracy (the product is defined for a non-symmetric H too)."""
    import copy
    import torch
    H0, _, _, _ = small_problem(3, 64, 0.3, 2064)
    H = copy.copy(H0)
    vals = H0.values.copy().reshape(H0.nblocks, H0.b, H0.b)
    scale = 10.0 ** np.linspace(-20, 20, H0.M)
    tile_row = np.repeat(np.arange(H0.M // H0.b), np.diff(H0.row_ptr))
    for p in range(H0.nblocks):
        vals[p] *= scale[tile_row[p] * H0.b:(tile_row[p] + 1) * H0.b, None]
    zr, dr = 5, 70                                            # global rows: all zero / diagonal only
    for p in range(H0.nblocks):
        I, J = tile_row[p], H0.col_idx[p]
        if I == zr // H0.b:
            vals[p][zr % H0.b, :] = 0.0
        if I == dr // H0.b:
            d = vals[p][dr % H0.b, dr % H0.b] if J == I else 0.0
            vals[p][dr % H0.b, :] = 0.0
            if J == I:
                vals[p][dr % H0.b, dr % H0.b] = d
    H.values = vals.reshape(H0.values.shape)
    rp, col, val = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    Hd = build_i8(tt, H, mode="i8x7")
    N = 96
    X = synth.dense_normal(H.M, N, 81)
    ref = oracle.spmm(rp, col, val, 1.0, X)
    Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
    tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
    got = Y.cpu().numpy()
    assert np.all(got[zr] == 0.0)
    rn = np.linalg.norm(ref, axis=1)
    rn[rn == 0] = 1.0
    assert np.max(np.linalg.norm(got - ref, axis=1) / rn) <= 10 * ACC["i8x7"]


def kohn_sham_like(b, seed):
    """A truncated Kohn-Sham-shaped H (couplings below 1e-4 Ha are dropped, the leading ones are O(1-10)):
    the generator's structure and zero mask (G = 3, z = 0.4), every kept entry of an OFF-DIAGONAL tile replaced by
    sign * 10^u, u ~ U[-4, 1], symmetric -- five orders of magnitude of dynamic range INSIDE every row of couplings."""
    import copy
    H0, _, _, _ = small_problem(3, b, 0.4, 2300 + b)
    rng = np.random.default_rng(seed)
    M = H0.M
    V = np.where(rng.random((M, M)) < 0.5, -1.0, 1.0) * 10.0 ** rng.uniform(-4.0, 1.0, (M, M))
    V = np.triu(V) + np.triu(V, 1).T
    vals = H0.values.copy().reshape(H0.nblocks, b, b)
    tile_row = np.repeat(np.arange(M // b), np.diff(H0.row_ptr))
    for p in range(H0.nblocks):
        I, J = int(tile_row[p]), int(H0.col_idx[p])
        if I != J:
            vals[p] = np.where(vals[p] != 0.0, V[I * b:(I + 1) * b, J * b:(J + 1) * b], 0.0)
    H = copy.copy(H0)
    H.values = vals.reshape(H0.values.shape)
    return H


@pytest.mark.parametrize("b", [64, 128])
def test_in_row_dynamic_range(tt, b):
    """The fixed-point operand format scales a whole row of H by ONE power of two: small couplings next to large ones keep
    fewer bits than fp64 gives them (K3 error bound n 2^-51 hmax_i ymax_j).  On rows spanning 1e-4 .. 1e1 the
    product must still meet north_star's 1e-12 and a degree-20 filter 1e-10, worst column within 10x, in both int8 modes."""
    import torch
    H = kohn_sham_like(b, 77)
    C = synth.bsr_to_csr_nonzeros(H)
    off = np.abs(C.values[np.abs(C.values) < 15.0])
    assert off.min() < 2e-4 and off.max() > 5.0              # the range is really there
    N, m = 150, 20
    v0 = synth.dense_normal(H.M, 1, 23, synth.STREAM_V0).reshape(-1)
    a0, bb, _ = oracle.lanczos_bounds(C.row_ptr, C.col_idx, C.values, v0, 40)
    a0, bb = a0 - 0.05 * (bb - a0), bb + 0.05 * (bb - a0)    # safely outside the spectrum (this H is far from the generator's)
    X = synth.dense_normal(H.M, N, 91)
    ref_mm = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, X)
    errs = {}
    for wide in (False, True):
        a, bb_, a0_ = bounds_for(a0, bb, N, H.M, wide=wide)
        ref_f = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, bb_, a0_)
        for mode in ("i8x7", "i8", "fp64"):
            Hd = build_i8(tt, H, mode="i8x7")
            Hd.set_math_mode({"i8x7": tt.MATH_I8X7, "i8": tt.MATH_I8, "fp64": tt.MATH_FP64}[mode])
            Y = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
            tt.spmm(Hd, 1.0, dev(X), 0.0, Y, use_work=True)
            e1, w1 = relerr(Y.cpu().numpy(), ref_mm), worst_col_relerr(Y.cpu().numpy(), ref_mm)
            tt.cheb_filter(Hd, dev(X), Y, m, a, bb_, a0_)
            e2, w2 = relerr(Y.cpu().numpy(), ref_f), worst_col_relerr(Y.cpu().numpy(), ref_f)
            errs[(mode, wide)] = (e1, w1, e2, w2)
            print(f"in-row dynamic range b={b} {mode} wide={wide}: spmm {e1:.2e} (worst col {w1:.2e}), filter {e2:.2e} ({w2:.2e})")
    for (mode, wide), (e1, w1, e2, w2) in errs.items():
        assert e1 <= TOL_SPMM and w1 <= 10 * TOL_SPMM, (mode, wide, e1, w1)
        assert e2 <= TOL_FILTER and w2 <= 10 * TOL_FILTER, (mode, wide, e2, w2)


@pytest.mark.parametrize("mode", ["i8x7", "i8"])
def test_degree20_wide_gap_b128(tt, mode):
    """SURVEY 8(d) "extra parity-only cases": the wide gap a = a0 + 0.25 (b - a0) with the headline degree m = 20
    (|T_20(t0)| ~ 1.7e9: the iterates shrink by nine orders of magnitude, column scales change every step) on 128-wide tiles."""
    import torch
    H, C, (rp, col, val), (a0, bb) = small_problem(3, 128, 0.4, 2128)
    N, m = 200, 20
    a, bb, a0 = bounds_for(a0, bb, N, H.M, wide=True)
    Hd = build_i8(tt, H, mode=mode)
    X = synth.dense_normal(H.M, N, 93)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)
    assert np.linalg.norm(ref) < 0.5 * np.linalg.norm(X)     # three quarters of the spectrum are damped by ~1e-9
    for inplace in (False, True):
        Xd = dev(X)
        Y = Xd if inplace else torch.empty_like(Xd)
        tt.cheb_filter(Hd, Xd, Y, m, a, bb, a0, panel_cols=128)
        got = Y.cpu().numpy()
        e, w = relerr(got, ref), worst_col_relerr(got, ref)
        print(f"m=20 wide gap b=128 {mode} inplace={inplace}: {e:.2e} worst col {w:.2e}")
        assert e <= TOL_FILTER and w <= 10 * TOL_FILTER


def _filter_with_env(tt, H, X, m, a, b, a0, env, mode="i8x7", panel=0):
    """Build (the handle reads the environment switches) and filter under the given environment."""
    import os
    import torch
    old = {k: os.environ.get(k) for k in env}
    os.environ.update(env)
    try:
        Hd = build_i8(tt, H, mode=mode)
    finally:
        for k, v in old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v
    Y = torch.empty(H.M, X.shape[1], dtype=torch.float64, device="cuda")
    tt.cheb_filter(Hd, dev(X), Y, m, a, b, a0, panel_cols=panel)
    return Y.cpu().numpy()


@pytest.mark.parametrize("G,b,N", [(3, 128, 200), (3, 64, 150), (2, 96, 100)])
@pytest.mark.parametrize("wide", [False, True])
def test_epilogue_digits_prediction_and_fallback(tt, G, b, N, wide):
    """From the second step on K3's epilogue writes the next iterate's digit planes itself with a PREDICTED column exponent
    (K3 "digits from the epilogue"); tiles whose prediction is outgrown are redone from the fp64 iterate.  The
    prediction path (default), the all-fallback path (bias -6: every prediction fails, i.e. the true exponents of the former
    design) and a pessimistic prediction (bias +3: three bits fewer) must all meet the filter tolerance."""
    H, C, (rp, col, val), (a0, bb) = small_problem(G, b, 0.4, 2400 + b)
    m = 12
    a, bb, a0 = bounds_for(a0, bb, N, H.M, wide=wide)
    X = synth.dense_normal(H.M, N, 97)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)
    for bias in ("0", "-6", "3"):
        got = _filter_with_env(tt, H, X, m, a, bb, a0, {"TTDFT_K3_PREDICT_BIAS": bias}, panel=128)
        e, w = relerr(got, ref), worst_col_relerr(got, ref)
        print(f"epilogue digits G={G} b={b} wide={wide} bias={bias}: {e:.2e} worst col {w:.2e}")
        assert e <= TOL_FILTER and w <= 10 * TOL_FILTER
        if bias != "3":
            assert e <= 50 * ACC["i8x7"]                      # no precision lost to the prediction beyond a guard bit or two


def test_column_that_grows_past_its_prediction(tt):
    """A column whose iterate nearly vanishes at step 1 and comes back at step 2 (X_j = e_i for a row i of H that holds only its
    diagonal entry c: (H - c) e_i = 0 up to rounding, then Y_2 = beta_1 X + ...): the predicted exponent of Y_2 is ~50 binary
    orders too small, the column's tile must be redone and the result still match the oracle; so must columns next to it."""
    import copy
    import torch
    H0, _, _, (a0, bb) = small_problem(3, 64, 0.3, 2064)
    N, m = 70, 10                                            # even degree: p_m(c) = +-1 / T_m(t0) != 0
    a, bb, a0 = bounds_for(a0, bb, N, H0.M)
    c = 0.5 * (a + bb)
    rows = [5, 700]                                          # rows that keep only their diagonal entry, set to c
    vals = H0.values.copy().reshape(H0.nblocks, H0.b, H0.b)
    tile_row = np.repeat(np.arange(H0.M // H0.b), np.diff(H0.row_ptr))
    for p in range(H0.nblocks):
        I, J = int(tile_row[p]), int(H0.col_idx[p])
        for r in rows:
            if I == r // H0.b:
                vals[p][r % H0.b, :] = 0.0
            if J == r // H0.b:
                vals[p][:, r % H0.b] = 0.0
            if I == J == r // H0.b:
                vals[p][r % H0.b, r % H0.b] = c
    H = copy.copy(H0)
    H.values = vals.reshape(H0.values.shape)
    rp, col, val = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    X = synth.dense_normal(H.M, N, 99)
    X[:, 3] = 0.0
    X[rows[0], 3] = 1.0                                      # column 3 = e_5; column 66 (ragged last tile) = 2 e_700
    X[:, 66] = 0.0
    X[rows[1], 66] = 2.0
    ref = oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)
    assert abs(ref[rows[0], 3]) > 1e-3                        # the column does come back
    for mode in ("i8x7", "i8"):
        got = _filter_with_env(tt, H, X, m, a, bb, a0, {}, mode=mode)
        e, w = relerr(got, ref), worst_col_relerr(got, ref)
        print(f"vanishing column {mode}: {e:.2e} worst col {w:.2e}")
        assert e <= TOL_FILTER and w <= 10 * TOL_FILTER


@pytest.mark.parametrize("mode", ["i8x7", "i8"])
@pytest.mark.parametrize("G,b,N", [(3, 96, 330), (2, 96, 100), (3, 64, 200), (3, 128, 257), (2, 128, 64)])
def test_transposed_kernel_k3t(tt, G, b, N, mode):
    """Kernel K3T (the tile's rows on the N axis of the MMA, columns of Y on M: the default for 96-wide tiles, TTDFT_K3_T=1
    elsewhere) against the oracle and against kernel K3 (TTDFT_K3_T=0): the integer sums and the epilogue arithmetic are the same,
    so the two kernels must agree bit for bit -- ragged column counts, single steps and whole filters."""
    import os
    import torch
    H, C, (rp, col, val), (a0, bb) = small_problem(G, b, 0.4, 2500 + b)
    m = 7
    a, bb, a0 = bounds_for(a0, bb, N, H.M, wide=True)
    X = synth.dense_normal(H.M, N, 101)
    Z = synth.dense_normal(H.M, N, 102)
    ref = oracle.cheb_filter(rp, col, val, X, m, a, bb, a0)
    ref_step = oracle.cheb_step(rp, col, val, 0.173, 9.5, -0.31, X, Z)
    out = {}
    for t in ("0", "1"):
        os.environ["TTDFT_K3_T"] = t
        try:
            Hd = build_i8(tt, H, mode=mode)
        finally:
            os.environ.pop("TTDFT_K3_T", None)
        Y = torch.full((H.M, N + 3), float("nan"), dtype=torch.float64, device="cuda")
        tt.cheb_filter(Hd, dev(X), Y[:, :N], m, a, bb, a0, panel_cols=256)
        O = torch.empty(H.M, N, dtype=torch.float64, device="cuda")
        tt.cheb_step(Hd, 0.173, 9.5, -0.31, dev(X), dev(Z), O, use_work=True)
        assert torch.isnan(Y[:, N:]).all()                    # nothing written outside the view
        out[t] = (Y[:, :N].cpu().numpy(), O.cpu().numpy())
        assert relerr(out[t][0], ref) <= TOL_FILTER and worst_col_relerr(out[t][0], ref) <= 10 * TOL_FILTER
        assert relerr(out[t][1], ref_step) <= ACC[mode]
    assert np.array_equal(out["0"][1], out["1"][1])
    full = N // 64 * 64          # K3 redoes a ragged last 64-column tile with the true exponents, K3T keeps the predicted ones there
    assert np.array_equal(out["0"][0][:, :full], out["1"][0][:, :full])
    assert relerr(out["0"][0], out["1"][0]) <= 1e-14
