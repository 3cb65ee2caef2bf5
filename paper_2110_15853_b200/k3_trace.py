"""Clock trace of kernel K3 (bsr_i8_kernel): where one CTA spends its cycles per work item.

    python -m paper_2110_15853_b200.k3_trace [--workload si] [--ncols 4096]

Uses the library's debug hook `ttdft_debug_k3_trace` (not part of include/ttdft.h): while a device buffer is registered,
every K3 launch records 8 clock64() stamps per work item of CTA 0 (first 512 items):
  [0] MMA warp: item start      [1] accumulators free (accempty)      [2] last MMA of the item committed
  [3] epilogue: ready           [4] accumulators complete (accfull)   [5] TMEM drained, released
  [6] output phase done         [7] tiles in the item's block row
The table below groups the items by tile count (27 = interior block row, 18 = face, 12 = edge, 8 = corner of the grid).
DESIGN.md "K3" quotes these numbers; profiles/r01d_k3_trace.md holds one run.
"""
from __future__ import annotations

import argparse
import ctypes
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="si")
    ap.add_argument("--ncols", type=int, default=4096)
    args = ap.parse_args()
    import torch
    import paper_2110_15853_b200 as tt

    cfg = synth.CONFIGS[args.workload]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    dev = torch.device("cuda")
    Hd = tt.h_build_bsr(H.M, H.b, *(torch.from_numpy(x).to(dev) for x in (H.row_ptr, H.col_idx, H.values)))
    Hd.set_math_mode(tt.MATH_I8X7)
    N = args.ncols
    X = torch.randn(cfg.M, N, dtype=torch.float64, device=dev)
    Z = torch.randn(cfg.M, N, dtype=torch.float64, device=dev)
    O = torch.empty_like(X)
    work = torch.empty(tt.step_work_bytes(Hd, N) + 16, dtype=torch.uint8, device=dev)
    for _ in range(2):
        tt.cheb_step(Hd, 0.1, 10.0, -0.2, X, Z, O, work=work)
    torch.cuda.synchronize()
    buf = torch.zeros(512 * 8, dtype=torch.int64, device=dev)
    lib = ctypes.CDLL(tt.library_path())
    lib.ttdft_debug_k3_trace.argtypes = [ctypes.c_void_p]
    lib.ttdft_debug_k3_trace(buf.data_ptr())
    tt.cheb_step(Hd, 0.1, 10.0, -0.2, X, Z, O, work=work)
    torch.cuda.synchronize()
    lib.ttdft_debug_k3_trace(None)
    t = buf.cpu().numpy().reshape(512, 8)
    rows = []
    for i in range(1, 512):
        s0, s1, s2, e3, e4, e5, e6, nj = t[i]
        if s0 == 0:
            break
        rows.append((nj, s1 - s0, s2 - s1, e4 - e3, e5 - e4, e6 - e5, e4 - s2))
    r = np.array(rows, dtype=np.float64)
    print("| tiles | items | MMA: wait for free accumulators | MMA: issue phase | per tile | epilogue: wait for accumulators | "
          "drain | output phase | epilogue late by | ideal MMA (3,584/tile) |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for nj in sorted(set(r[:, 0])):
        m = r[r[:, 0] == nj].mean(0)
        print(f"| {int(nj)} | {int((r[:, 0] == nj).sum())} | {m[1]:.0f} | {m[2]:.0f} | {m[2] / nj:.0f} | {m[3]:.0f} | {m[4]:.0f} | "
              f"{m[5]:.0f} | {m[6]:.0f} | {nj * 3584:.0f} |")


if __name__ == "__main__":
    main()
