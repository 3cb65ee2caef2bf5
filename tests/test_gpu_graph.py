"""The filter is stream-asynchronous with no host synchronisation inside (SURVEY.md 8(b) "all work is enqueued on the given stream
and the call returns without synchronising"), so a whole `ttdft_cheb_filter` call -- every fused step, digit pass and buffer rotation --
can be captured into ONE CUDA graph and replayed: the launch-bound small problems (BASELINE.json config 1) then cost one graph launch.
Replays must give the eager call's bits and match the oracle, also after the input buffer's contents change."""
import numpy as np
import pytest

import oracle
import synth
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


@pytest.mark.parametrize("G,b,z,N,m", [(4, 32, 0.0, 32, 10), (3, 64, 0.3, 96, 6), (2, 128, 0.4, 200, 5)])
def test_filter_captured_in_a_cuda_graph(tt, G, b, z, N, m):
    import torch
    H, C, _, (a0, bb) = small_problem(G, b, z, 9300 + b)
    a, bq, a0q = bounds_for(a0, bb, N, H.M)
    Hd = tt.h_build_bsr(H.M, H.b, dev(H.row_ptr), dev(H.col_idx), dev(H.values))
    X1, X2 = synth.dense_normal(H.M, N, 94), synth.dense_normal(H.M, N, 95)
    Xd = dev(X1)
    Yd = torch.empty_like(Xd)
    work = torch.empty(tt.cheb_filter_work_bytes(Hd, N) + 1024, dtype=torch.uint8, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):                                  # warm-up on the side stream (function attributes, tensor maps)
        tt.cheb_filter(Hd, Xd, Yd, m, a, bq, a0q, work=work)
    s.synchronize()
    eager = Yd.clone()
    n0 = tt.launch_count()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        tt.cheb_filter(Hd, Xd, Yd, m, a, bq, a0q, work=work)
    launches = tt.launch_count() - n0
    assert launches >= m
    Yd.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(Yd, eager)                               # the replay's bits are the eager call's
    assert relerr(Yd.cpu().numpy(), oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X1, m, a, bq, a0q)) <= 1e-10
    Xd.copy_(dev(X2))                                           # new wavefunctions in the same buffer
    g.replay()
    torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, X2, m, a, bq, a0q)) <= 1e-10
    # timing, informational: eager launches vs one graph launch
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    torch.cuda.synchronize()
    e0.record()
    for _ in range(20):
        tt.cheb_filter(Hd, Xd, Yd, m, a, bq, a0q, work=work)
    e1.record()
    for _ in range(20):
        g.replay()
    e2.record()
    torch.cuda.synchronize()
    print(f"\nfilter G={G} b={b} N={N} m={m}: {launches} kernels; eager {e0.elapsed_time(e1) / 20 * 1e3:.1f} us, graph replay {e1.elapsed_time(e2) / 20 * 1e3:.1f} us")
