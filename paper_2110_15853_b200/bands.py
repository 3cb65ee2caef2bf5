"""Column-band parallelism ("band parallelization": the wavefunction block is cut into column groups G_p and H is
replicated per group).  Columns are independent through the whole filter, so a band needs NO collective on the data
path: every rank filters its own columns with its replica of H.  This module holds only the index arithmetic and the two
control-plane reductions bench.py and a multi-GPU driver need (max-over-ranks time, gathering the bands for the next ChFSI step);
it works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def band_of(rank: int, world: int, ncols: int) -> tuple[int, int]:
    """(first column, number of columns) of rank's band when `ncols` columns are cut into `world` bands (strong scaling):
    tau = ncols // world columns each, the first ncols % world ranks get one more (the paper's partition rule, L244-248, applied
    to columns)."""
    if world < 1 or not (0 <= rank < world) or ncols < 0:
        raise ValueError("bad band arguments")
    tau, nu = divmod(ncols, world)
    first = rank * tau + min(rank, nu)
    return first, tau + (1 if rank < nu else 0)


def weak_band(rank: int, ncols_per_rank: int) -> tuple[int, int]:
    """(first column, number of columns) of rank's band when every rank owns `ncols_per_rank` columns of a global block of
    world * ncols_per_rank columns (weak scaling: what bench.py --gpus N times)."""
    return rank * ncols_per_rank, ncols_per_rank


def max_over_ranks(seconds: float, device=None) -> float:
    """The slowest rank's time (the job's time); no-op without an initialised process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_bands(Y_band, ncols_total: int):
    """All ranks' filtered bands side by side: the M x ncols_total block the next ChFSI step (orthonormalisation) needs.
    Y_band: this rank's M x n_r tensor (row-major).  Returns an M x ncols_total tensor on every rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return Y_band
    world, rank = dist.get_world_size(), dist.get_rank()
    M = Y_band.shape[0]
    out = torch.empty((M, ncols_total), dtype=Y_band.dtype, device=Y_band.device)
    c0, n = band_of(rank, world, ncols_total)
    if tuple(Y_band.shape) != (M, n):
        raise ValueError(f"rank {rank} owns {n} columns, got {Y_band.shape[1]}")
    nmax = band_of(0, world, ncols_total)[1]              # all_gather wants equal pieces: pad the narrower bands by one column
    mine = torch.zeros((M, nmax), dtype=Y_band.dtype, device=Y_band.device)
    mine[:, :n] = Y_band
    pieces = [torch.empty((M, nmax), dtype=Y_band.dtype, device=Y_band.device) for _ in range(world)]
    dist.all_gather(pieces, mine)
    for r in range(world):
        c0, n = band_of(r, world, ncols_total)
        out[:, c0:c0 + n] = pieces[r][:, :n]
    return out
