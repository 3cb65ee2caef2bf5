"""Writes tests/golden/bounds.json: the spectral bounds (a, b, a0) handed to the filter for each
BASELINE.json config.  The paper takes eps_0, eps_ub^w, eps_ub^uw as inputs of Algorithm 1
 and defers how they are obtained to [30, 31] (L232); reading #5:
30-step oracle Lanczos with residual-corrected Ritz bounds, a = a0 + (N/M)(b - a0).

This script calls only synth/ (inputs) and oracle/ (Lanczos).  Nothing from the CUDA path.
Usage: python tests/golden/make_bounds.py [tiny al si largest]
"""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import oracle  # noqa: E402
import synth  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "bounds.json")


def main():
    names = sys.argv[1:] or list(synth.CONFIGS)
    data = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            data = json.load(f)
    for name in names:
        cfg = synth.CONFIGS[name]
        t0 = time.time()
        H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
        C = synth.bsr_to_csr_nonzeros(H)
        nblocks = H.nblocks
        del H
        v0 = synth.dense_normal(cfg.M, 1, cfg.seed, synth.STREAM_V0).reshape(-1)
        a0, b, info = oracle.lanczos_bounds(C.row_ptr, C.col_idx, C.values, v0, 30)
        a = a0 + (cfg.N / cfg.M) * (b - a0)
        data[name] = {
            "a": a, "b": b, "a0": a0, "nnz": C.nnz, "nblocks": nblocks, "M": cfg.M, "N": cfg.N,
            "theta_min": float(info["theta"][0]), "theta_max": float(info["theta"][-1]),
            "recipe": "oracle.lanczos_bounds(k=30, v0=synth STREAM_V0) ; a = a0 + (N/M)(b-a0)",
        }
        print(name, data[name], f"{time.time() - t0:.1f}s", flush=True)
        with open(OUT, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
