"""The N > 1 path on CPU: world_size-2 gloo processes run the band arithmetic and the two control-plane reductions of
paper_2110_15853_b200/bands.py, with the CPU oracle standing in for the per-rank filter (no GPU here).  Column independence of the
filter (oracle pin P5) makes the gathered bands equal to the single-process result bit for bit."""
import os
import socket

import numpy as np
import pytest

import oracle
import synth
from paper_2110_15853_b200 import bands


def test_band_partition_covers_every_column_once():
    for ncols in (0, 1, 7, 64, 4096, 14336):
        for world in (1, 2, 3, 8):
            seen = np.zeros(ncols, int)
            sizes = []
            for r in range(world):
                c0, n = bands.band_of(r, world, ncols)
                seen[c0:c0 + n] += 1
                sizes.append(n)
            assert np.all(seen == 1)
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)   # first ranks get the extra column
    assert bands.weak_band(3, 4096) == (3 * 4096, 4096)
    with pytest.raises(ValueError):
        bands.band_of(2, 2, 10)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ncols, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = synth.CONFIGS["tiny"]
        H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
        C = synth.bsr_to_csr_nonzeros(H)
        a, b, a0 = 2.0, 22.0, -1.0
        c0, n = bands.band_of(rank, world, ncols)
        Xb = np.empty((cfg.M, n))
        synth.dense_normal(cfg.M, n, cfg.seed, synth.STREAM_X, col0=c0, out=Xb)       # this rank's columns of the global block
        Yb = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, Xb, 5, a, b, a0)      # the per-rank filter (oracle stands in)
        Y = bands.gather_bands(torch.from_numpy(Yb), ncols)
        t = bands.max_over_ranks(1.0 + rank)
        np.save(os.path.join(out_dir, f"Y{rank}.npy"), Y.numpy())
        np.save(os.path.join(out_dir, f"t{rank}.npy"), np.array([t]))
    finally:
        dist.destroy_process_group()


def test_two_rank_band_filter_equals_single_process(tmp_path):
    import torch.multiprocessing as mp
    world, ncols = 2, 11                      # 6 + 5 columns
    port = _free_port()
    mp.spawn(_worker, args=(world, port, ncols, str(tmp_path)), nprocs=world, join=True)
    cfg = synth.CONFIGS["tiny"]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    C = synth.bsr_to_csr_nonzeros(H)
    X = np.empty((cfg.M, ncols))
    synth.dense_normal(cfg.M, ncols, cfg.seed, synth.STREAM_X, col0=0, out=X)
    ref = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X, 5, 2.0, 22.0, -1.0)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"Y{r}.npy"), ref)                   # every rank holds the whole filtered block
        assert np.load(tmp_path / f"t{r}.npy")[0] == 2.0                              # the slowest rank's time
