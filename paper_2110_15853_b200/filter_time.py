"""Whole-filter time of BASELINE.json's other configs (2 "al", 4 "largest": parity-test cases, not bench lines) in both math modes:

    python -m paper_2110_15853_b200.filter_time al largest

X ~ N(0,1) generated on the device (in place for config 4, whose X is 45 GB), one timed ttdft_cheb_filter call after a 2-step warm-up,
CUDA events, per-kernel launch times from the library's own event pairs.  Prints one JSON line per (config, math mode)."""
import os, sys, json
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import numpy as np


def main():
    import torch
    import synth
    import paper_2110_15853_b200 as tt
    dev = torch.device("cuda")
    for wl in sys.argv[1:]:
        cfg = synth.CONFIGS[wl]
        d = json.load(open(os.path.join(ROOT, "tests", "golden", "bounds.json")))[wl]
        a, b, a0 = d["a"], d["b"], d["a0"]
        H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
        nnz = int(np.count_nonzero(H.values))
        Hd = tt.h_build_bsr(H.M, H.b, *(torch.from_numpy(x).to(dev) for x in (H.row_ptr, H.col_idx, H.values)))
        del H
        X = torch.randn(cfg.M, cfg.N, dtype=torch.float64, device=dev)
        panel = cfg.panel if cfg.panel else 0
        for mode, name in ((tt.MATH_I8X7, "i8x7"), (tt.MATH_FP64, "fp64")):
            Hd.set_math_mode(mode)
            work = torch.empty(tt.cheb_filter_work_bytes(Hd, cfg.N, panel) + 16, dtype=torch.uint8, device=dev)
            inplace = cfg.M * cfg.N * 8 > 30e9
            Y = X if inplace else torch.empty_like(X)
            reps = 1 if inplace else 2
            tt.cheb_filter(Hd, X, Y, 2, a, b, a0, panel_cols=panel, work=work)   # warm-up (2 steps)
            torch.cuda.synchronize()
            for k in tt.KERNEL_IDS: tt.timing_read(k)
            tt.timing_enable(True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps): tt.cheb_filter(Hd, X, Y, cfg.m, a, b, a0, panel_cols=panel, work=work)
            e1.record(); torch.cuda.synchronize()
            tt.timing_enable(False)
            kt = {k: tt.timing_read(k) for k in tt.KERNEL_IDS}
            t = e0.elapsed_time(e1) / reps
            if inplace: X.normal_()
            print(json.dumps({"workload": wl, "M": cfg.M, "N": cfg.N, "b": cfg.b, "m": cfg.m, "panel": panel, "mode": name, "inplace": inplace,
                              "filter_ms": t, "useful_tflops": 2.0 * nnz * cfg.N * cfg.m / t / 1e9,
                              "kernels_ms_each": {k: round(v[0] / max(v[1], 1), 3) for k, v in kt.items() if v[1]}}), flush=True)
            del work
        del X, Y, Hd
        torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
