"""Row partition of H (paper_2110_15853_b200/rows.py) on ONE GPU: the slab handles
of 2 and 3 emulated ranks run one after the other (no kernel waits on another), their row slabs are put together, and the result
must equal the full handle's step BIT FOR BIT (every row's sum runs over the same tiles in the same order) and the oracle within
north_star's tolerance -- on the fp64 tensor-core kernel and on the int8 kernel (slab handles have EMPTY block rows there)."""
import numpy as np
import pytest

import oracle
import synth
from paper_2110_15853_b200 import rows
from util import bounds_for, relerr, small_problem

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


def handles(tt, H, world):
    out = []
    nb = H.M // H.b
    for r in range(world):
        I0, n = rows.slab_of(r, world, nb)
        rp, ci, va = rows.slab_bsr(H.row_ptr, H.col_idx, H.values, I0, n)
        out.append((I0 * H.b, (I0 + n) * H.b, tt.h_build_bsr(H.M, H.b, dev(rp), dev(ci), dev(va))))
    return out


@pytest.mark.parametrize("G,b,z,world,use_work", [(3, 32, 0.0, 2, False), (3, 64, 0.3, 2, True), (3, 64, 0.3, 3, False),
                                                   (3, 128, 0.4, 3, True), (2, 96, 0.4, 3, True)])
def test_slab_steps_equal_full_step_bit_for_bit(tt, G, b, z, world, use_work):
    import torch
    H, C, _, _ = small_problem(G, b, z, 9100 + b)
    Hf = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    N = 70
    Yk, Ykm1 = dev(synth.dense_normal(H.M, N, 91)), dev(synth.dense_normal(H.M, N, 92))
    alpha, c, beta = 0.37, 9.5, -0.81
    full = torch.empty_like(Yk)
    tt.cheb_step(Hf, alpha, c, beta, Yk, Ykm1, full, use_work=use_work)
    ref = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, alpha, c, beta, Yk.cpu().numpy(), Ykm1.cpu().numpy())
    assert relerr(full.cpu().numpy(), ref) <= 1e-12
    got = torch.full_like(Yk, float("nan"))
    for r0, r1, Hs in handles(tt, H, world):
        part = torch.empty_like(Yk)
        tt.cheb_step(Hs, alpha, c, beta, Yk, Ykm1, part, use_work=use_work)
        got[r0:r1] = part[r0:r1]
    assert torch.equal(got, full)


def test_row_sharded_filter_lockstep_emulation(tt):
    """cheb_filter_rows as rank 0 of 3 would run it; the exchange is emulated by running the other ranks' slab steps right there."""
    import torch
    G, b, z = 3, 64, 0.3
    H, C, _, (a0, bb) = small_problem(G, b, z, 9200)
    N, m = 48, 7
    a, bq, a0q = bounds_for(a0, bb, N, H.M)
    X = synth.dense_normal(H.M, N, 93)
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, m, a, bq, a0q)
    hs = handles(tt, H, 3)
    last = {}

    def step(alpha, c, beta, Yk, Ykm1, Yout):
        last["args"] = (alpha, c, beta, Yk, None if Ykm1 is None else Ykm1.clone())       # Yout may alias Ykm1
        tt.cheb_step(hs[0][2], alpha, c, beta, Yk, Ykm1, Yout, use_work=True)
        Yout[hs[0][1]:] = float("nan")

    def exchange(Yout, block, nb):
        alpha, c, beta, Yk, Ykm1 = last["args"]
        for r0, r1, Hs in hs[1:]:
            part = torch.empty_like(Yk)
            tt.cheb_step(Hs, alpha, c, beta, Yk, Ykm1, part, use_work=True)
            Yout[r0:r1] = part[r0:r1]
        return Yout

    c, alpha, beta = tt.cheb_scalars(m, a, bq, a0q)
    Xd = dev(X)
    Y = rows.cheb_filter_rows(step, Xd, m, c, alpha, beta, b, H.M // b, exchange=exchange)
    assert torch.equal(Xd, dev(X))                                                         # X not modified
    assert relerr(Y.cpu().numpy(), ref) <= 1e-10
    # and the library's own single-GPU filter gives the same bits
    Hf = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    Yf = torch.empty_like(Xd)
    tt.cheb_filter(Hf, Xd, Yf, m, a, bq, a0q)
    assert relerr(Y.cpu().numpy(), Yf.cpu().numpy()) <= 1e-13


@pytest.mark.parametrize("G,b,world,mode", [(4, 32, 2, "fp64"), (4, 64, 2, "fp64"), (4, 64, 2, "i8x7"), (4, 96, 2, "i8x7")])
def test_interior_and_boundary_handles(tt, G, b, world, mode):
    """The overlapped row partition runs two handles per rank, built with TTDFT_OWNED_ROWS_ONLY: interior block rows (tiles only
    inside the slab) and boundary ones.  Each step writes ONLY the rows of its own block rows, so both go into the same output:
    together they equal the full handle's step bit for bit on the slab and leave every other row untouched; the interior step of
    the fp64 kernel reads no row outside the slab (remote rows poisoned with NaN).  The int8 modes scale by whole-column maxima,
    i.e. they need the complete iterate and are not eligible for the overlap -- they are only checked on complete data here."""
    import torch
    H, C, _, _ = small_problem(G, b, 0.3, 9300 + b)
    nb = H.M // H.b
    MODE = {"fp64": tt.MATH_FP64, "i8x7": tt.MATH_I8X7}[mode]
    Hf = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values)).set_math_mode(MODE)
    N = 40
    Yk, Ykm1 = dev(synth.dense_normal(H.M, N, 94)), dev(synth.dense_normal(H.M, N, 95))
    alpha, c, beta = 0.37, 9.5, -0.81
    full = torch.empty_like(Yk)
    tt.cheb_step(Hf, alpha, c, beta, Yk, Ykm1, full, use_work=True)
    for r in range(world):
        I0, n = rows.slab_of(r, world, nb)
        (rpi, cii, vai), (rpb, cib, vab), mask = rows.split_slab(H.row_ptr, H.col_idx, H.values, I0, n)
        assert 0 < mask.sum() < n
        Hi = tt.h_build_bsr(H.M, H.b, dev(rpi), dev(cii), dev(vai), flags=tt.OWNED_ROWS_ONLY).set_math_mode(MODE)
        Hb = tt.h_build_bsr(H.M, H.b, dev(rpb), dev(cib), dev(vab), flags=tt.OWNED_ROWS_ONLY).set_math_mode(MODE)
        Yin = Yk.clone()
        if mode == "fp64":
            Yin[:I0 * b] = float("nan")
            Yin[(I0 + n) * b:] = float("nan")
        for use_work in ([True, False] if mode == "fp64" else [True]):
            out = torch.full_like(Yk, float("nan"))
            tt.cheb_step(Hi, alpha, c, beta, Yin, Ykm1, out, use_work=use_work)
            rows_i = torch.zeros(H.M, dtype=torch.bool, device="cuda")
            rows_i[I0 * b:(I0 + n) * b] = dev(np.repeat(mask, b))
            assert torch.equal(out[rows_i], full[rows_i]) and torch.isnan(out[~rows_i]).all()
            tt.cheb_step(Hb, alpha, c, beta, Yk, Ykm1, out, use_work=use_work)
            assert torch.equal(out[I0 * b:(I0 + n) * b], full[I0 * b:(I0 + n) * b])
            assert torch.isnan(out[:I0 * b]).all() and torch.isnan(out[(I0 + n) * b:]).all()
    # the generic kernel (CSR) honours the flag per row
    Cs = synth.bsr_to_csr_nonzeros(H)
    keep = np.zeros(H.M, bool)
    keep[: H.M // 3] = True
    counts = np.where(keep, np.diff(Cs.row_ptr), 0)
    rp = np.zeros(H.M + 1, np.int32)
    np.cumsum(counts, out=rp[1:])
    nk = int(rp[-1])
    Hc = tt.h_build_csr(H.M, dev(rp), dev(Cs.col_idx[:nk]), dev(Cs.values[:nk]), flags=tt.OWNED_ROWS_ONLY)
    out = torch.full_like(Yk, float("nan"))
    tt.cheb_step(Hc, alpha, c, beta, Yk, Ykm1, out)
    ref = oracle.cheb_step(Cs.row_ptr, Cs.col_idx, Cs.values, alpha, c, beta, Yk.cpu().numpy(), Ykm1.cpu().numpy())
    assert relerr(out[: H.M // 3].cpu().numpy(), ref[: H.M // 3]) <= 1e-12 and torch.isnan(out[H.M // 3:]).all()
