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
