"""Row partition of H across GPUs ("the Hamiltonian matrix and the wavefunction matrix are partitioned row-wise",
L244-248 the partition rule, L258 "regardless of the implementation, collective communication over either X or X' will be needed";
SURVEY.md 8(e), 8(f)-3).  Needed only when H does not fit one GPU -- none of BASELINE.json's configs: their multi-GPU path is the
collective-free column bands of bands.py.

Rank k owns a contiguous slab of block rows [I0, I0 + nI) of the tile format (whole subdomains, so every tile belongs to exactly one
rank) and builds its handle from the M x M matrix that holds only those block rows.  One recurrence step is then
    Y_{k+1}[rows of rank r] = fused step of rank r's handle on the full iterates           (the library's kernels, unchanged)
    all-gather of the row slabs                                                              (the collective over X' of L258)
The paper's own variant sums transposed slab products, Y = sum_k (H_k)^T X_k (Eq. 22), and all-reduces the M x N result
through the host; it moves the same M x N x 8 bytes per step as the all-gather here, but its sum must be complete before the
recurrence's scale/shift/axpby can be applied, which would split the fused epilogue off into a second pass.  With the all-gather
every output row is finished by the rank that owns it, the step stays ONE kernel, and the result is bit-identical to the
single-GPU step (each row's sum runs over the same tiles in the same order).

This module is index arithmetic plus the exchange; it works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def slab_of(rank: int, world: int, nb: int) -> tuple[int, int]:
    """(first block row, number of block rows) of rank's slab: tau = nb // world each, the first nb % world ranks one more
    (applied to block rows so that no subdomain is split)."""
    if world < 1 or not (0 <= rank < world) or nb < 0:
        raise ValueError("bad slab arguments")
    tau, nu = divmod(nb, world)
    return rank * tau + min(rank, nu), tau + (1 if rank < nu else 0)


def slab_bsr(row_ptr: np.ndarray, col_idx: np.ndarray, values: np.ndarray, I0: int, nI: int):
    """BSR arrays of the M x M matrix that keeps only block rows [I0, I0 + nI) of (row_ptr, col_idx, values): the other block
    rows are empty.  col_idx and values are views (no copy of the tiles)."""
    nb = len(row_ptr) - 1
    if not (0 <= I0 and 0 <= nI and I0 + nI <= nb):
        raise ValueError("slab outside the matrix")
    lo, hi = int(row_ptr[I0]), int(row_ptr[I0 + nI])
    rp = (np.clip(np.asarray(row_ptr, np.int64), lo, hi) - lo).astype(np.int32)
    return rp, col_idx[lo:hi], values[lo:hi]


def all_gather_rows(Y, block: int, nb: int):
    """Completes Y (M x n, row-major, full width) in place: the row slab of every rank r is taken from rank r.
    One broadcast per rank on the contiguous slab (slabs may differ by one block row, which all_gather's equal pieces cannot hold)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return Y
    world = dist.get_world_size()
    for r in range(world):
        I0, nI = slab_of(r, world, nb)
        if nI:
            dist.broadcast(Y[I0 * block:(I0 + nI) * block], src=r)
    return Y


def cheb_filter_rows(step, X, m: int, c: float, alpha, beta, block: int, nb: int, exchange=all_gather_rows):
    """Algorithm 1 step 1 with H partitioned by rows.
    step(alpha_k, c, beta_k, Yk, Ykm1 or None, Yout): one fused recurrence step of THIS rank's slab handle (ttdft_cheb_step); it
    must fill at least this rank's rows of Yout.  X: the full M x n block on every rank (not modified).  c, alpha, beta: the
    scalars of ttdft_cheb_scalars.  Returns the full filtered block on every rank (X itself for m = 0)."""
    if m == 0:
        return X
    import torch
    bufs = [torch.empty_like(X), torch.empty_like(X)]
    Yk, Ykm1 = X, None
    for k in range(m):
        # A4: from the third step on the oldest iterate's buffer takes the new one (it is read elementwise at the output position)
        out = bufs[k] if k < 2 else Ykm1
        step(float(alpha[k]), float(c), float(beta[k]) if k > 0 else 0.0, Yk, Ykm1, out)
        exchange(out, block, nb)
        Yk, Ykm1 = out, Yk
    return Yk
