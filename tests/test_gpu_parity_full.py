"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot filter 4,096-14,336 columns of a 2-4e5-row H in reasonable time, so:
  * a seeded column sample (first/last column of every panel + random ones) is compared element by
    element -- exact, because columns are independent through the whole filter;
  * EVERY column is covered by the self-adjointness (Freivalds-style) identity
        <u, F(X)[:, j]> = <F(u), X[:, j]>    (F = p_m(H) is symmetric)
    with F(u) computed by the oracle for r seeded Gaussian probes u.
Every arithmetic mode of the library (fp64 DMMA, int8 digit planes x7 / x6) runs against the same
oracle values and the same tolerance.
"""
import json
import os

import numpy as np
import pytest

import oracle
import synth
from util import relerr, worst_col_relerr

pytestmark = pytest.mark.gpu

TOL_FILTER = 1e-10
BOUNDS = os.path.join(os.path.dirname(__file__), "golden", "bounds.json")


def bounds(name):
    with open(BOUNDS) as f:
        d = json.load(f)[name]
    return d["a"], d["b"], d["a0"], d["nnz"]


def run_full(name, nsample, nprobe, inplace):
    import torch
    import paper_2110_15853_b200 as tt
    cfg = synth.CONFIGS[name]
    a, b, a0, nnz_expected = bounds(name)
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    C = synth.bsr_to_csr_nonzeros(H)
    assert C.nnz == nnz_expected                      # same matrix the stored bounds were computed for
    Hd = tt.h_build_bsr(H.M, H.b, torch.from_numpy(H.row_ptr).cuda(), torch.from_numpy(H.col_idx).cuda(),
                        torch.from_numpy(H.values).cuda())
    assert Hd.info()["kernel"] == 1
    del H
    # X on the device, generated on the host in column chunks (counter-based: any chunking gives the same X)
    Xd = torch.empty((cfg.M, cfg.N), dtype=torch.float64, device="cuda")
    chunk = 1024
    for c0 in range(0, cfg.N, chunk):
        w = min(chunk, cfg.N - c0)
        Xd[:, c0:c0 + w] = torch.from_numpy(synth.dense_normal(cfg.M, w, cfg.seed, synth.STREAM_X, col0=c0)).cuda()
    # oracle inputs: sampled columns regenerated from the generator, plus Gaussian probes
    cols = synth.column_sample(cfg.N, cfg.panel, nsample, cfg.seed)
    Xs = np.empty((cfg.M, len(cols)))
    for k, c in enumerate(cols):
        synth.dense_normal(cfg.M, 1, cfg.seed, synth.STREAM_X, col0=int(c), out=Xs[:, k:k + 1])
    assert np.array_equal(Xd[:, torch.from_numpy(cols).cuda()].cpu().numpy(), Xs)
    U = synth.dense_normal(cfg.M, nprobe, cfg.seed, synth.STREAM_U)
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, np.hstack([Xs, U]), cfg.m, a, b, a0)
    ref_s, FU = ref[:, :len(cols)], ref[:, len(cols):]
    FtX = (torch.from_numpy(FU).cuda().T @ Xd).cpu().numpy()        # <F(u), X_j>, before X may be overwritten

    Ud = torch.from_numpy(U).cuda()
    unorm = np.linalg.norm(U, axis=0)
    cols_d = torch.from_numpy(cols).cuda()
    modes = [("fp64", tt.MATH_FP64)]
    if Hd.info()["i8_planes"]:
        modes += [("i8x7", tt.MATH_I8X7), ("i8", tt.MATH_I8)]
    X0 = Xd.clone() if (inplace and len(modes) > 1) else None     # in place overwrites X: restore it per mode
    Yd = Xd if inplace else torch.empty_like(Xd)
    for k, (mname, mode) in enumerate(modes):
        if inplace and k > 0:
            Xd.copy_(X0)
        elif not inplace:
            Yd.fill_(float("nan"))
        Hd.set_math_mode(mode)
        assert Hd.info()["math"] == mode
        tt.cheb_filter(Hd, Xd, Yd, cfg.m, a, b, a0, panel_cols=cfg.panel)
        torch.cuda.synchronize()
        got = Yd[:, cols_d].cpu().numpy()
        e_f, e_c = relerr(got, ref_s), worst_col_relerr(got, ref_s)
        UtY = (Ud.T @ Yd).cpu().numpy()
        ynorm = torch.linalg.vector_norm(Yd, dim=0).cpu().numpy()
        adj = np.abs(UtY - FtX) / (unorm[:, None] * ynorm[None, :])
        print(f"{name}/{mname}: sample relerr {e_f:.2e} worst col {e_c:.2e}; adjoint check max {adj.max():.2e} "
              f"over {cfg.N} columns")
        assert np.isfinite(ynorm).all()
        assert e_f <= TOL_FILTER and e_c <= 10 * TOL_FILTER
        assert adj.max() <= TOL_FILTER


def test_full_config2_al():
    run_full("al", nsample=32, nprobe=4, inplace=False)


def test_full_config3_si_headline():
    run_full("si", nsample=32, nprobe=4, inplace=False)


def test_full_config4_largest_inplace_panels():
    run_full("largest", nsample=32, nprobe=4, inplace=True)


def test_config5_sweep_points():
    """BASELINE.json config 5 at full size with an oracle comparison at the points sweep.py times: config 3's H (M = 221,184) as
    subdomain-ordered BSR (tile kernels, every math mode) and as the seeded symmetrically permuted CSR without labels (generic
    kernel K2: nnz = 3.98e8, the 64-bit offsets a small case never reaches), one ttdft_spmm and one ttdft_cheb_step each.
    N = 16 and 256: EVERY element against the oracle (12.7 / 204 GFLOP of oracle work).  N = 4,096 (BSR): a seeded column sample
    element by element (columns are independent in one product) plus the Freivalds identity u^T (H X) = (H u)^T X over all columns."""
    import torch
    import paper_2110_15853_b200 as tt
    TOL = 1e-12
    cfg = synth.CONFIGS["si"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    C = synth.bsr_to_csr_nonzeros(H)
    dev = torch.device("cuda")
    Hb = tt.h_build_bsr(H.M, H.b, torch.from_numpy(H.row_ptr).to(dev), torch.from_numpy(H.col_idx).to(dev),
                        torch.from_numpy(H.values).to(dev))
    del H
    perm = synth.permutation(cfg.M, cfg.seed + 50)               # the permutation sweep.py uses
    Cp = synth.permute_csr(C, perm)
    Hc = tt.h_build_csr(Cp.M, torch.from_numpy(Cp.row_ptr).to(dev), torch.from_numpy(Cp.col_idx).to(dev),
                        torch.from_numpy(Cp.values).to(dev), flags=tt.CHECK_SORTED)
    assert Hb.info()["kernel"] == 1 and Hc.info()["kernel"] == 0 and Hc.info()["nnz_stored"] == C.nnz
    alpha, c, beta = 0.1, 10.0, -0.2                             # the step sweep.py times
    modes = [("fp64", tt.MATH_FP64), ("i8x7", tt.MATH_I8X7), ("i8", tt.MATH_I8)]

    def check(tag, got, ref):
        e, w = relerr(got, ref), worst_col_relerr(got, ref)
        print(f"config5 {tag}: relerr {e:.2e} worst column {w:.2e}")
        assert e <= TOL and w <= 10 * TOL, (tag, e, w)

    for N in (16, 256):
        X = synth.dense_normal(cfg.M, N, cfg.seed + N, synth.STREAM_X)
        Z = synth.dense_normal(cfg.M, N, cfg.seed + N + 1, synth.STREAM_X)
        ref_mm = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, X)
        ref_st = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, alpha, c, beta, X, Z)
        Xd, Zd = torch.from_numpy(X).to(dev), torch.from_numpy(Z).to(dev)
        O = torch.empty_like(Xd)
        for mname, mode in modes:
            Hb.set_math_mode(mode)
            O.fill_(float("nan"))
            tt.spmm(Hb, 1.0, Xd, 0.0, O, use_work=True)
            check(f"bsr/{mname} spmm N={N}", O.cpu().numpy(), ref_mm)
            O.fill_(float("nan"))
            tt.cheb_step(Hb, alpha, c, beta, Xd, Zd, O, use_work=True)
            check(f"bsr/{mname} step N={N}", O.cpu().numpy(), ref_st)
        # permuted CSR: H' = P H P^T on X' = P X gives P Y (reading #12)
        Xp, Zp = synth.permute_rows(X, perm), synth.permute_rows(Z, perm)
        Xd, Zd = torch.from_numpy(Xp).to(dev), torch.from_numpy(Zp).to(dev)
        O.fill_(float("nan"))
        tt.spmm(Hc, 1.0, Xd, 0.0, O)
        check(f"csr/K2 spmm N={N}", O.cpu().numpy(), synth.permute_rows(ref_mm, perm))
        O.fill_(float("nan"))
        tt.cheb_step(Hc, alpha, c, beta, Xd, Zd, O)
        check(f"csr/K2 step N={N}", O.cpu().numpy(), synth.permute_rows(ref_st, perm))
        del Xd, Zd, O
    del Hc, Cp

    # N = 4,096 on the tile kernels: sampled columns + Freivalds over all columns
    N = 4096
    Xd = torch.empty((cfg.M, N), dtype=torch.float64, device=dev)
    Zd = torch.empty((cfg.M, N), dtype=torch.float64, device=dev)
    for c0 in range(0, N, 1024):
        Xd[:, c0:c0 + 1024] = torch.from_numpy(synth.dense_normal(cfg.M, 1024, cfg.seed, synth.STREAM_X, col0=c0)).to(dev)
        Zd[:, c0:c0 + 1024] = torch.from_numpy(synth.dense_normal(cfg.M, 1024, cfg.seed + 7, synth.STREAM_X, col0=c0)).to(dev)
    cols = synth.column_sample(N, 0, 24, cfg.seed)
    cols_d = torch.from_numpy(cols).to(dev)
    Xs, Zs = Xd[:, cols_d].cpu().numpy(), Zd[:, cols_d].cpu().numpy()
    U = synth.dense_normal(cfg.M, 3, cfg.seed, synth.STREAM_U)
    ref_mm = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, Xs)
    ref_st = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, alpha, c, beta, Xs, Zs)
    HU = oracle.spmm(C.row_ptr, C.col_idx, C.values, 1.0, U)        # H symmetric: u^T (H X) = (H u)^T X
    Ud, HUd = torch.from_numpy(U).to(dev), torch.from_numpy(HU).to(dev)
    want = (HUd.T @ Xd).cpu().numpy()
    scale = np.linalg.norm(HU, axis=0)[:, None] * torch.linalg.vector_norm(Xd, dim=0).cpu().numpy()[None, :]
    O = torch.empty_like(Xd)
    for mname, mode in modes:
        Hb.set_math_mode(mode)
        O.fill_(float("nan"))
        tt.spmm(Hb, 1.0, Xd, 0.0, O, use_work=True)
        check(f"bsr/{mname} spmm N={N} (sample)", O[:, cols_d].cpu().numpy(), ref_mm)
        fre = np.abs((Ud.T @ O).cpu().numpy() - want) / scale
        print(f"config5 bsr/{mname} spmm N={N}: Freivalds max {fre.max():.2e}")
        assert fre.max() <= TOL
        O.fill_(float("nan"))
        tt.cheb_step(Hb, alpha, c, beta, Xd, Zd, O, use_work=True)
        check(f"bsr/{mname} step N={N} (sample)", O[:, cols_d].cpu().numpy(), ref_st)
        assert torch.isfinite(O).all()
