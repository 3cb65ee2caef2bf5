"""Row partition of H (paper_2110_15853_b200/rows.py) on CPU: the slab arithmetic,
and world_size-2 gloo processes that each own a slab of block rows, with the CPU oracle's single step standing in for the per-rank
fused step (no GPU here).  Every row's sum runs over the same entries in the same order as in the unpartitioned matrix, so the
row-sharded filter equals the single-process oracle filter bit for bit."""
import os
import socket

import numpy as np
import pytest

import oracle
import synth
from paper_2110_15853_b200 import rows


def test_slab_partition_and_slab_matrix():
    for nb in (0, 1, 5, 64, 1728, 4096):
        for world in (1, 2, 3, 8):
            seen = np.zeros(nb, int)
            sizes = []
            for r in range(world):
                I0, n = rows.slab_of(r, world, nb)
                seen[I0:I0 + n] += 1
                sizes.append(n)
            assert np.all(seen == 1) and max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        rows.slab_of(3, 3, 10)
    H = synth.hamiltonian_bsr(3, 8, 0.3, 77)
    full = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    X = synth.dense_normal(H.M, 3, 78)
    ref = oracle.spmm(*full, 1.0, X)
    acc = np.zeros_like(ref)
    for r in range(4):
        I0, n = rows.slab_of(r, 4, (H.M // H.b))
        rp, ci, va = rows.slab_bsr(H.row_ptr, H.col_idx, H.values, I0, n)
        assert len(rp) == (H.M // H.b) + 1 and rp[0] == 0 and rp[-1] == len(ci) == len(va)
        part = oracle.spmm(*oracle.bsr_to_csr(H.b, rp, ci, va), 1.0, X)
        assert np.array_equal(part[I0 * H.b:(I0 + n) * H.b], ref[I0 * H.b:(I0 + n) * H.b])      # the slab's rows, bit for bit
        mask = np.ones(H.M, bool)
        mask[I0 * H.b:(I0 + n) * H.b] = False
        assert not part[mask].any()                                                              # nothing outside them
        acc += part
    assert np.array_equal(acc, ref)
    with pytest.raises(ValueError):
        rows.slab_bsr(H.row_ptr, H.col_idx, H.values, (H.M // H.b), 1)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


A, B, A0, DEG, NCOLS = 2.0, 22.0, -1.0, 6, 5


def _scalars(m, a, b, a0):
    """Algorithm 1's scalars, restated for the test: alpha_k, beta_k of step k."""
    e, c = (b - a) / 2.0, (b + a) / 2.0
    sigma = e / (a0 - c)
    sigma1 = sigma
    gamma = 2.0 / sigma1
    alpha, beta = [sigma1 / e], [0.0]
    for _ in range(2, m + 1):
        sigma2 = 1.0 / (gamma - sigma)
        alpha.append(2.0 * sigma2 / e)
        beta.append(-(sigma * sigma2))
        sigma = sigma2
    return c, alpha, beta


def test_interior_boundary_split():
    """The interior block rows of a slab (every tile's block column inside the slab) and the boundary ones partition the slab;
    the two matrices built from them add up to the slab's matrix bit for bit."""
    H = synth.hamiltonian_bsr(4, 8, 0.3, 79)                              # 64 block rows, 16 per z-layer of the 4 x 4 x 4 grid
    nb = H.M // H.b
    X = synth.dense_normal(H.M, 3, 80)
    for world in (2, 3, 4):
        total_interior = 0
        for r in range(world):
            I0, n = rows.slab_of(r, world, nb)
            (rpi, cii, vai), (rpb, cib, vab), mask = rows.split_slab(H.row_ptr, H.col_idx, H.values, I0, n)
            rp, ci, va = rows.slab_bsr(H.row_ptr, H.col_idx, H.values, I0, n)
            assert mask.shape == (n,) and len(cii) + len(cib) == len(ci)
            slab = oracle.spmm(*oracle.bsr_to_csr(H.b, rp, ci, va), 1.0, X)
            inner = oracle.spmm(*oracle.bsr_to_csr(H.b, rpi, cii, vai), 1.0, X)
            outer = oracle.spmm(*oracle.bsr_to_csr(H.b, rpb, cib, vab), 1.0, X)
            rows_i = np.repeat(mask, H.b)
            assert np.array_equal(inner[I0 * H.b:(I0 + n) * H.b][rows_i], slab[I0 * H.b:(I0 + n) * H.b][rows_i])
            assert np.array_equal(outer[I0 * H.b:(I0 + n) * H.b][~rows_i], slab[I0 * H.b:(I0 + n) * H.b][~rows_i])
            assert not inner[I0 * H.b:(I0 + n) * H.b][~rows_i].any() and not outer[I0 * H.b:(I0 + n) * H.b][rows_i].any()
            # interior rows reference only columns inside the slab
            for i in np.nonzero(mask)[0]:
                cols = H.col_idx[H.row_ptr[I0 + i]:H.row_ptr[I0 + i + 1]]
                assert cols.min() >= I0 and cols.max() < I0 + n
            total_interior += int(mask.sum())
        assert total_interior < nb
        if world == 2:
            assert total_interior == 32                                   # slabs of two x-layers: the outer layer of each is interior


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        H = synth.hamiltonian_bsr(3, 16, 0.3, 4242)                       # 27 block rows: slabs of 14 and 13
        I0, n = rows.slab_of(rank, world, (H.M // H.b))
        rp, ci, va = rows.slab_bsr(H.row_ptr, H.col_idx, H.values, I0, n)
        Cs = oracle.bsr_to_csr(H.b, rp, ci, va)                           # this rank's slab as an M x M CSR (other rows empty)
        X = synth.dense_normal(H.M, NCOLS, 4243)

        def step(alpha, c, beta, Yk, Ykm1, Yout):                         # the per-rank fused step (oracle stands in)
            res = oracle.cheb_step(*Cs, alpha, c, beta, Yk.numpy(), None if Ykm1 is None else Ykm1.numpy())
            Yout.copy_(torch.from_numpy(res))
            Yout[:I0 * H.b] = float("nan")                                # rows of other ranks must come from the exchange
            Yout[(I0 + n) * H.b:] = float("nan")

        c, alpha, beta = _scalars(DEG, A, B, A0)
        Y = rows.cheb_filter_rows(step, torch.from_numpy(X.copy()), DEG, c, alpha, beta, H.b, (H.M // H.b))
        np.save(os.path.join(out_dir, f"Y{rank}.npy"), Y.numpy())

        # the overlapped form: interior block rows step while the previous exchange is in flight, boundary rows after it.  The
        # remote rows of every new iterate are poisoned until the exchange delivers them, so an interior step that touched them
        # (or a boundary step that ran too early) would leave NaNs behind.
        H = synth.hamiltonian_bsr(4, 8, 0.3, 4244)                        # 64 block rows: slabs of two x-layers, one of them interior
        I0, n = rows.slab_of(rank, world, (H.M // H.b))
        X = synth.dense_normal(H.M, NCOLS, 4245)
        (rpi, cii, vai), (rpb, cib, vab), mask = rows.split_slab(H.row_ptr, H.col_idx, H.values, I0, n)
        assert mask.sum() == 16
        Ci, Cb = oracle.bsr_to_csr(H.b, rpi, cii, vai), oracle.bsr_to_csr(H.b, rpb, cib, vab)
        rows_i = np.zeros(H.M, bool)
        rows_i[I0 * H.b:(I0 + n) * H.b] = np.repeat(mask, H.b)
        rows_b = np.zeros(H.M, bool)
        rows_b[I0 * H.b:(I0 + n) * H.b] = np.repeat(~mask, H.b)

        def make_step(Cx, sel, poison):
            def f(alpha, c, beta, Yk, Ykm1, Yout):
                yk = Yk.numpy().copy()
                if poison:                                                # interior rows must not read another rank's rows
                    yk[:I0 * H.b] = float("nan")
                    yk[(I0 + n) * H.b:] = float("nan")
                    yk[np.isnan(yk)] = 1e300                              # 0 * NaN would survive in the oracle's sums: use a huge value
                res = oracle.cheb_step(*Cx, alpha, c, beta, yk, None if Ykm1 is None else Ykm1.numpy())
                out = Yout.numpy()
                out[sel] = res[sel]
                if poison:
                    out[:I0 * H.b] = float("nan")
                    out[(I0 + n) * H.b:] = float("nan")
            return f

        Y2 = rows.cheb_filter_rows(make_step(Ci, rows_i, True), torch.from_numpy(X.copy()), DEG, c, alpha, beta, H.b, (H.M // H.b),
                                   step_boundary=make_step(Cb, rows_b, False))
        np.save(os.path.join(out_dir, f"Z{rank}.npy"), Y2.numpy())
    finally:
        dist.destroy_process_group()


def test_two_rank_row_sharded_filter_equals_single_process(tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    H = synth.hamiltonian_bsr(3, 16, 0.3, 4242)
    full = oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values)
    X = synth.dense_normal(H.M, NCOLS, 4243)
    ref = oracle.cheb_filter(*full, X, DEG, A, B, A0)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"Y{r}.npy"), ref)       # every rank holds the whole filtered block, bit for bit
    H = synth.hamiltonian_bsr(4, 8, 0.3, 4244)
    ref = oracle.cheb_filter(*oracle.bsr_to_csr(H.b, H.row_ptr, H.col_idx, H.values), synth.dense_normal(H.M, NCOLS, 4245), DEG, A, B, A0)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"Z{r}.npy"), ref)       # ... also with interior steps overlapping the exchange
