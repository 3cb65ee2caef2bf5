"""Row partition of H across GPUs ("the Hamiltonian matrix and the wavefunction matrix are partitioned row-wise",
L244-248 the partition rule, L258 "regardless of the implementation, collective communication over either X or X' will be needed";
SURVEY.md 8(e), 8(f)-3).  Needed only when H does not fit one GPU -- none of BASELINE.json's configs: their multi-GPU path is the
collective-free column bands of bands.py.

Rank k owns a contiguous slab of block rows [I0, I0 + nI) of the tile format (whole subdomains, so every tile belongs to exactly one
rank) and builds its handle(s) from the M x M matrix that holds only those block rows.  One recurrence step is then
    Y_{k+1}[rows of rank r] = fused step of rank r's handle on the full iterates           (the library's kernels; a handle built
                              with TTDFT_OWNED_ROWS_ONLY writes only the rows of its own block rows)
    all-gather of the row slabs                                                              (the collective over X' of L258)
as ONE collective per step (all_gather_into_tensor: in place on the iterate when the slabs are equal, through one padded staging
buffer when they differ by a block row), issued asynchronously so that it overlaps the next step's INTERIOR block rows -- those
whose tiles multiply only rows this rank computed itself; the BOUNDARY block rows (a tile reaches into another rank's slab) wait
for it.  On a 3-D grid of subdomains cut into slabs the boundary is two layers of G^2 block rows per rank, the interior the rest.
The overlap is for TTDFT_MATH_FP64 handles: the int8 modes scale every column of the iterate by its maximum over ALL rows, so their
step needs the complete iterate (pass one handle and no step_boundary there).

Why an all-gather and not the paper's reduction.  The paper sums transposed slab products, Y = sum_k (H_k)^T X_k (Eq. 22),
and all-reduces the M x N result through the host.  That moves the same M x N x 8 bytes per rank and step, but the sum must be
complete before the recurrence's scale, shift and axpby can be applied, which would split the fused epilogue off into a second
pass over the iterate -- and a floating-point reduction across ranks changes the summation order with the rank count.  With the
all-gather every output row is finished by the rank that owns it, the step stays ONE kernel per row subset, and the result is
bit-identical to the single-GPU step (each row's sum runs over the same tiles in the same order) for any number of ranks.

This module is index arithmetic plus the exchange; it works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
Unmeasured on hardware: one GPU per call in this pool.
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


def interior_mask(row_ptr: np.ndarray, col_idx: np.ndarray, I0: int, nI: int) -> np.ndarray:
    """mask[i] for block row I0 + i of the slab: True if every tile of the block row has its block column inside the slab, i.e. the
    row's step reads only rows of the iterate this rank computed itself and need not wait for the exchange."""
    rp = np.asarray(row_ptr, np.int64)
    ci = np.asarray(col_idx)
    mask = np.zeros(nI, bool)
    for i in range(nI):
        cols = ci[rp[I0 + i]:rp[I0 + i + 1]]
        mask[i] = bool(np.all((cols >= I0) & (cols < I0 + nI)))
    return mask


def subset_bsr(row_ptr: np.ndarray, col_idx: np.ndarray, values: np.ndarray, keep: np.ndarray):
    """BSR arrays of the M x M matrix that keeps only the block rows with keep[I] (any subset; the tiles are copied in order)."""
    rp = np.asarray(row_ptr, np.int64)
    nb = len(rp) - 1
    keep = np.asarray(keep, bool)
    if keep.shape != (nb,):
        raise ValueError("keep must have one entry per block row")
    counts = np.where(keep, rp[1:] - rp[:-1], 0)
    new_rp = np.zeros(nb + 1, np.int64)
    np.cumsum(counts, out=new_rp[1:])
    sel = np.concatenate([np.arange(rp[I], rp[I + 1]) for I in np.nonzero(keep)[0]]) if keep.any() else np.zeros(0, np.int64)
    return new_rp.astype(np.int32), np.ascontiguousarray(np.asarray(col_idx)[sel]), np.ascontiguousarray(np.asarray(values)[sel])


def split_slab(row_ptr: np.ndarray, col_idx: np.ndarray, values: np.ndarray, I0: int, nI: int):
    """(interior BSR, boundary BSR, interior mask) of the slab [I0, I0 + nI): two M x M matrices whose block rows partition the
    slab's.  Build one handle from each; interior steps overlap the exchange, boundary steps follow it."""
    nb = len(row_ptr) - 1
    m = interior_mask(row_ptr, col_idx, I0, nI)
    keep_i = np.zeros(nb, bool)
    keep_b = np.zeros(nb, bool)
    keep_i[I0:I0 + nI] = m
    keep_b[I0:I0 + nI] = ~m
    return subset_bsr(row_ptr, col_idx, values, keep_i), subset_bsr(row_ptr, col_idx, values, keep_b), m


class _Pending:
    """An exchange in flight: wait() makes the caller's stream (NCCL) or thread (gloo) wait for it and finishes the unpacking."""

    def __init__(self, work=None, after=None):
        self.work, self.after = work, after

    def wait(self):
        if self.work is not None:
            self.work.wait()
            self.work = None
        if self.after is not None:
            self.after()
            self.after = None


def all_gather_rows_async(Y, block: int, nb: int, stage=None) -> _Pending:
    """Starts the completion of Y (M x n, row-major, full width, contiguous): the row slab of every rank r is taken from rank r.
    ONE collective.  Equal slabs: in place (all_gather_into_tensor with the local slab as the input).  Slabs that differ by a
    block row: every rank sends its slab padded to the largest one into `stage` (world x rows_max x n, allocated if None) and the
    pieces are copied into place by wait().  Y's local slab must be complete (on the current stream) when this is called."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return _Pending()
    world, rank = dist.get_world_size(), dist.get_rank()
    slabs = [slab_of(r, world, nb) for r in range(world)]
    I0, nI = slabs[rank]
    n = Y.shape[1]
    if not Y.is_contiguous():
        raise ValueError("all_gather_rows needs a contiguous iterate")
    if nb % world == 0:
        return _Pending(dist.all_gather_into_tensor(Y, Y[I0 * block:(I0 + nI) * block], async_op=True))
    rows_max = max(s[1] for s in slabs) * block
    if stage is None:
        stage = torch.empty((world + 1, rows_max, n), dtype=Y.dtype, device=Y.device)
    send, recv = stage[world], stage[:world]
    send[:nI * block].copy_(Y[I0 * block:(I0 + nI) * block])
    work = dist.all_gather_into_tensor(recv.view(world * rows_max, n), send, async_op=True)

    def unpack():
        for r, (J0, nJ) in enumerate(slabs):
            if r != rank and nJ:
                Y[J0 * block:(J0 + nJ) * block].copy_(recv[r, :nJ * block])

    return _Pending(work, unpack)


def all_gather_rows(Y, block: int, nb: int, stage=None):
    """Completes Y in place (blocking form of all_gather_rows_async)."""
    all_gather_rows_async(Y, block, nb, stage).wait()
    return Y


def cheb_filter_rows(step, X, m: int, c: float, alpha, beta, block: int, nb: int, exchange=None, step_boundary=None,
                     exchange_async=all_gather_rows_async):
    """Algorithm 1 step 1 with H partitioned by rows.
    step(alpha_k, c, beta_k, Yk, Ykm1 or None, Yout): one fused recurrence step of THIS rank's slab handle (ttdft_cheb_step); it
    must fill at least this rank's rows of Yout.  With step_boundary given, `step` is the INTERIOR handle's step (block rows that
    read only this rank's rows of Yk) and step_boundary the BOUNDARY handle's: the interior step of iteration k runs while the
    exchange of iteration k - 1 is still in flight, the boundary step after it has arrived.
    X: the full M x n block on every rank (not modified).  c, alpha, beta: the scalars of ttdft_cheb_scalars.
    exchange(Yout, block, nb): a blocking exchange (overrides exchange_async; used by the one-GPU emulation tests).
    Returns the full filtered block on every rank (X itself for m = 0)."""
    if m == 0:
        return X
    import torch
    bufs = [torch.empty_like(X), torch.empty_like(X)]
    Yk, Ykm1 = X, None
    pending = _Pending()
    for k in range(m):
        # A4: from the third step on the oldest iterate's buffer takes the new one (it is read elementwise at the output position)
        out = bufs[k] if k < 2 else Ykm1
        a_k, b_k = float(alpha[k]), (float(beta[k]) if k > 0 else 0.0)
        if step_boundary is None:
            pending.wait()
            step(a_k, float(c), b_k, Yk, Ykm1, out)
        else:
            step(a_k, float(c), b_k, Yk, Ykm1, out)            # interior rows: local data only, overlaps the exchange of Yk
            pending.wait()                                     # Yk's remote rows have arrived
            step_boundary(a_k, float(c), b_k, Yk, Ykm1, out)
        if exchange is not None:
            exchange(out, block, nb)
            pending = _Pending()
        else:
            pending = exchange_async(out, block, nb)
        Yk, Ykm1 = out, Yk
    pending.wait()
    return Yk
