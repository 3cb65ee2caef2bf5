"""One pass of Algorithm 1 (ChFSI) composed from the library's calls -- a usage example and an
end-to-end check, not a new kernel:

    step 1  ttdft_cheb_filter      X~  = p_m(H) X                      (the hot path)
    step 2  ttdft_orthonormalize   X_F = Orth(X~)                      (8(f)-2)
    step 3  ttdft_project          H_F = X_F^T H X_F                   (8(f)-1)
    step 4  torch.linalg.eigh      H_F Q = Q Lambda                    (n x n dense symmetric eigenproblem: the ONE library call;
                                                                        "library-shaped" in SURVEY.md 8(f)-4, not implemented here)
    step 5  ttdft_rotate           Psi = X_F Q                         (8(f)-4)

Everything of size M x n runs in the library's CUDA kernels; PyTorch allocates the buffers and solves the n x n problem.
"""
from __future__ import annotations

from . import api


def chfsi_iteration(H: "api.Hamiltonian", X, m: int, a: float, b: float, a0: float, panel_cols: int = 0):
    """Returns (Psi, Lambda): Psi M x n with orthonormal columns spanning the filtered subspace, rotated to the Ritz vectors;
    Lambda the n Ritz values in ascending order.  X: M x n float64 CUDA tensor (not modified)."""
    import torch
    M, n = X.shape
    Xf = torch.empty_like(X)
    api.cheb_filter(H, X, Xf, m, a, b, a0, panel_cols=panel_cols)          # step 1
    Xo = torch.empty_like(X)
    api.orthonormalize(Xf, Xo, passes=2)                                   # step 2
    del Xf
    HF = torch.empty((n, n), dtype=torch.float64, device=X.device)
    api.project(H, Xo, HF)                                                 # step 3
    lam, Q = torch.linalg.eigh(HF)                                         # step 4 (library; reads the lower triangle of H_F only)
    Psi = torch.empty_like(X)
    api.rotate(Xo, Q.contiguous(), Psi)                                    # step 5
    return Psi, lam


def bounds(H: "api.Hamiltonian", k: int = 30, seed: int = 0):
    """(a0, b): lower and upper bound of the spectrum by k Lanczos steps on the GPU (ttdft_lanczos_bounds) from a seeded start vector."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    v0 = torch.randn(H.M, dtype=torch.float64, device="cuda", generator=g)
    a0, b, _ = api.lanczos_bounds(H, v0, k)
    return a0, b


def chfsi(H: "api.Hamiltonian", X, m: int, b: float, a0: float, iterations: int, a: float | None = None):
    """`iterations` passes of Algorithm 1 with the usual bound update between passes (the paper takes the bounds as inputs and
    refers to [30, 31]): the filter damps [a, b]; after every pass a = largest Ritz value (the upper edge of the wanted
    spectrum), a0 = smallest Ritz value.  Returns (Psi, Lambda) of the last pass."""
    lam = None
    for _ in range(iterations):
        if lam is not None:
            a = float(lam[-1])
            a0 = min(a0, float(lam[0]))
        if a is None:
            a = a0 + (b - a0) * X.shape[1] / X.shape[0]
        if not (a0 < a < b):
            a = a0 + 1e-3 * (b - a0)
        X, lam = chfsi_iteration(H, X, m, a, b, a0)
    return X, lam


def main():
    """python -m paper_2110_15853_b200.chfsi [workload]: two passes of Algorithm 1 at the workload's shape (default config 3 "si"),
    every step timed with CUDA events (torch's current stream is the stream the library launches on here)."""
    import json
    import os
    import sys
    import torch
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    import synth
    name = sys.argv[1] if len(sys.argv) > 1 else "si"
    cfg = synth.CONFIGS[name]
    d = json.load(open(os.path.join(root, "tests", "golden", "bounds.json")))[name]
    a, b, a0 = d["a"], d["b"], d["a0"]
    dev = torch.device("cuda")
    Hs = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    H = api.h_build_bsr(Hs.M, Hs.b, *(torch.from_numpy(x).to(dev) for x in (Hs.row_ptr, Hs.col_idx, Hs.values)))
    del Hs
    M, n = cfg.M, cfg.N
    X = torch.randn(M, n, dtype=torch.float64, device=dev)
    for rep in range(2):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
        ev[0].record()
        Xf = torch.empty_like(X)
        api.cheb_filter(H, X, Xf, cfg.m, a, b, a0)
        ev[1].record()
        Xo = torch.empty_like(X)
        api.orthonormalize(Xf, Xo, passes=2)
        ev[2].record()
        del Xf
        HF = torch.empty((n, n), dtype=torch.float64, device=dev)
        api.project(H, Xo, HF)
        ev[3].record()
        lam, Q = torch.linalg.eigh(0.5 * (HF + HF.T))
        ev[4].record()
        Psi = torch.empty_like(X)
        api.rotate(Xo, Q.contiguous(), Psi)
        ev[5].record()
        torch.cuda.synchronize()
        t = [ev[i].elapsed_time(ev[i + 1]) for i in range(5)]
        print(json.dumps({"workload": name, "pass": rep + 1, "filter_ms": t[0], "orthonormalize_ms": t[1], "project_ms": t[2],
                          "eigh_torch_ms": t[3], "rotate_ms": t[4], "pass_ms": sum(t), "ritz_min": float(lam[0]), "ritz_max": float(lam[-1])}),
              flush=True)
        X = Psi
        del Xo, HF, Q


if __name__ == "__main__":
    main()
