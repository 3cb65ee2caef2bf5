"""BASELINE.json config 5: a single H*X (ttdft_spmm) and a single fused recurrence step
(ttdft_cheb_step) on config 3's H at N in {16, 64, 256, 1024, 4096}, in two layouts --
subdomain-ordered BSR and CSR with rows/columns symmetrically permuted by seed (irregular-access
stress; once as given -> generic kernel, once with the subdomain index of every row -> h_build regroups the rows
into tiles and the *_ws calls gather / scatter around the tile kernel; `csr+recovered`: no labels given, the library recovers
them from the sparsity pattern first) -- each reported against the binding roofline:
    T_roof = max(alg_bytes / BW_hbm, useful_flops / P_fp64).
The BSR layout runs three times: fp64 tensor-core MMA (kernel 1) and int8 digit planes (kernel 3 with 7 and 6 planes, through
the *_ws entry points; its time includes the digit extraction of X); roofline_frac > 1 there means
the fp64-accurate product ran faster than the native fp64 pipe could.

    python -m paper_2110_15853_b200.sweep [--workload si] [--layouts bsr,csr] [--out gpurun_out/sweep.json]

`--filter al,largest` instead times one whole ttdft_cheb_filter call on BASELINE.json's other configs (2 "al", 4 "largest":
parity-test cases, not bench lines) in the i8x7 and fp64 math modes: X ~ N(0,1) generated on the device (in place for config 4,
whose X is 45 GB), one timed call after a 2-step warm-up, CUDA events, per-kernel launch times from the library's own event pairs;
one JSON line per (config, math mode).
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

FP64_PEAK = 148 * 64 * 2 * 1.965e9        # flop/s, derived


def hbm_peak() -> float:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f)["hbm_gbs"] * 1e9
    return 6.65e12                            # B200_PROFILING.md fallback


def time_launches(fn, reps, flush):
    import torch
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush.zero_()                     # > L2 write between timed launches
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e-3)
    return float(np.median(ts)), float(np.min(ts))


def filter_times(workloads):
    """Whole-filter time of the named configs in both math modes (one JSON line each)."""
    import torch
    import paper_2110_15853_b200 as tt
    dev = torch.device("cuda")
    for wl in workloads:
        cfg = synth.CONFIGS[wl]
        with open(os.path.join(ROOT, "tests", "golden", "bounds.json")) as f:
            d = json.load(f)[wl]
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
            for k in tt.KERNEL_IDS:
                tt.timing_read(k)
            tt.timing_enable(True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                tt.cheb_filter(Hd, X, Y, cfg.m, a, b, a0, panel_cols=panel, work=work)
            e1.record()
            torch.cuda.synchronize()
            tt.timing_enable(False)
            kt = {k: tt.timing_read(k) for k in tt.KERNEL_IDS}
            t = e0.elapsed_time(e1) / reps
            if inplace:
                X.normal_()
            print(json.dumps({"workload": wl, "M": cfg.M, "N": cfg.N, "b": cfg.b, "m": cfg.m, "panel": panel, "mode": name,
                              "inplace": inplace, "filter_ms": t, "useful_tflops": 2.0 * nnz * cfg.N * cfg.m / t / 1e9,
                              "kernels_ms_each": {k: round(v[0] / max(v[1], 1), 3) for k, v in kt.items() if v[1]}}), flush=True)
            del work
        del X, Y, Hd
        torch.cuda.empty_cache()


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--filter", default="", help="comma-separated configs (al, largest): time one whole filter each instead of the sweep")
    ap.add_argument("--workload", default="si")
    ap.add_argument("--layouts", default="bsr,csr,csr+labels,csr+recovered")
    ap.add_argument("--ns", default="16,64,256,1024,4096")
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--csr-max-n", type=int, default=4096)
    ap.add_argument("--math", default="fp64,i8x7,i8", help="arithmetic of the bsr layout: fp64 (DMMA), i8x7 / i8 (7 / 6 digit planes)")
    ap.add_argument("--out", default="")
    return ap.parse_args(argv)


def main(argv=None, check=None):
    """check(permuted: bool, op, alpha_c_beta, X, Z, O) -> relative error of O against a reference, or None: a hook for the caller
    (bench.py --sweep passes one that runs the CPU oracle on a column sample; this module itself never touches the oracle)."""
    args = parse_args(argv)
    if args.filter:
        return filter_times(args.filter.split(","))
    import torch
    import paper_2110_15853_b200 as tt

    cfg = synth.CONFIGS[args.workload]
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    nnz = int(np.count_nonzero(H.values))
    bw = hbm_peak()
    dev = torch.device("cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    rows = []
    handles = {}
    if "bsr" in args.layouts:
        handles["bsr"] = tt.h_build_bsr(H.M, H.b, torch.from_numpy(H.row_ptr).to(dev), torch.from_numpy(H.col_idx).to(dev),
                                        torch.from_numpy(H.values).to(dev))
    mats = {}
    if check is not None and "bsr" in args.layouts:
        mats[False] = synth.bsr_to_csr_nonzeros(H)
    if "csr" in args.layouts:
        C = mats.get(False) or synth.bsr_to_csr_nonzeros(H)
        perm = synth.permutation(H.M, cfg.seed + 50)
        Cp = synth.permute_csr(C, perm)
        if check is not None:
            mats[True] = Cp
        del C
        rp_d, ci_d, va_d = (torch.from_numpy(Cp.row_ptr).to(dev), torch.from_numpy(Cp.col_idx).to(dev),
                            torch.from_numpy(Cp.values).to(dev))
        handles["csr"] = tt.h_build_csr(Cp.M, rp_d, ci_d, va_d)
        if "csr+labels" in args.layouts:
            # the same permuted CSR plus the subdomain index of every row: h_build regroups the rows into tiles (A0)
            labels = np.empty(Cp.M, np.int32)
            labels[perm] = (np.arange(Cp.M) // cfg.b).astype(np.int32)
            handles["csr+labels-i8x7"] = tt.h_build_csr(Cp.M, rp_d, ci_d, va_d, subdomain_of_row=torch.from_numpy(labels).to(dev))
            assert handles["csr+labels-i8x7"].info()["reordered"] == 1
        if "csr+recovered" in args.layouts:
            # the same permuted CSR WITHOUT labels: ttdft_recover_subdomains finds the subdomains from the sparsity pattern
            # (reading #18), then the labelled build as above
            import time
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            rec, n_groups = tt.recover_subdomains(Cp.M, rp_d, ci_d)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            assert n_groups == cfg.M // cfg.b, n_groups
            handles["csr+recovered-i8x7"] = tt.h_build_csr(Cp.M, rp_d, ci_d, va_d, subdomain_of_row=rec)
            torch.cuda.synchronize()
            t2 = time.perf_counter()
            inf = handles["csr+recovered-i8x7"].info()
            assert inf["reordered"] == 1 and inf["block"] == cfg.b
            truth = np.empty(Cp.M, np.int32)
            truth[perm] = (np.arange(Cp.M) // cfg.b).astype(np.int32)
            got = rec.cpu().numpy()
            first = np.full(n_groups, Cp.M, np.int64)
            np.minimum.at(first, truth, np.arange(Cp.M))
            same = bool(np.array_equal(np.argsort(np.argsort(first))[truth], got))   # planted groups numbered by their smallest row
            print(json.dumps({"recover_subdomains_s": t1 - t0, "labelled_build_s": t2 - t1, "n_groups": n_groups,
                              "equals_planted_partition": same, "nblocks": inf["nblocks"]}), flush=True)
            assert same
        del rp_d, ci_d, va_d
        if check is None:
            del Cp
    maths = args.math.split(",")
    if "bsr" in handles and handles["bsr"].info()["i8_planes"]:
        # the same handle through the int8 digit-plane kernel (ttdft_*_ws entry points), 7 and 6 planes
        if "i8x7" in maths:
            handles["bsr-i8x7"] = handles["bsr"]
        if "i8" in maths:
            handles["bsr-i8"] = handles["bsr"]
    if "fp64" not in maths:
        handles.pop("bsr", None)
    stored = {k: h.info()["nnz_stored"] for k, h in handles.items()}
    del H
    for N in [int(x) for x in args.ns.split(",")]:
        X = torch.randn(cfg.M, N, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(N))
        Z = torch.randn(cfg.M, N, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(N + 1))
        O = torch.empty_like(X)
        for layout, Hd in handles.items():
            if layout == "csr" and N > args.csr_max_n:
                continue
            i8 = layout.endswith("-i8") or layout.endswith("-i8x7")
            work = None
            if layout != "csr":
                Hd.set_math_mode({"bsr": tt.MATH_FP64, "bsr-i8": tt.MATH_I8, "bsr-i8x7": tt.MATH_I8X7,
                                  "csr+labels-i8x7": tt.MATH_I8X7,
                                  "csr+recovered-i8x7": tt.MATH_I8X7}[layout])
            if i8:
                work = torch.empty(tt.step_work_bytes(Hd, N) + 16, dtype=torch.uint8, device=dev)
            for op in ("spmm", "step"):
                if op == "spmm":
                    fn = lambda: tt.spmm(Hd, 1.0, X, 0.0, O, work=work)
                    alg_bytes = 8.0 * nnz + 16.0 * cfg.M * N
                    coeffs = (1.0, 0.0, 0.0)
                else:
                    fn = lambda: tt.cheb_step(Hd, 0.1, 10.0, -0.2, X, Z, O, work=work)
                    alg_bytes = 8.0 * nnz + 24.0 * cfg.M * N
                    coeffs = (0.1, 10.0, -0.2)
                reps = args.reps if (layout == "bsr" or N <= 256) else 3
                t_med, t_min = time_launches(fn, reps, flush)
                flops = 2.0 * nnz * N
                t_roof = max(alg_bytes / bw, flops / FP64_PEAK)
                row = {"layout": layout, "op": op, "N": N, "ms": t_med * 1e3, "ms_min": t_min * 1e3,
                       "useful_tflops": flops / t_med / 1e12, "alg_gbs": alg_bytes / t_med / 1e9,
                       "executed_tflops": 2.0 * stored[layout] * N / t_med / 1e12,
                       "binds": "hbm" if alg_bytes / bw > flops / FP64_PEAK else "fp64",
                       "roofline_frac": t_roof / t_med, "kernel": 3 if i8 else Hd.info()["kernel"]}
                if check is not None:
                    row["relerr"] = check(mats[layout.startswith("csr")], op, coeffs, X, Z, O)
                rows.append(row)
                print(json.dumps(row), flush=True)
        del X, Z, O
    out = {"workload": args.workload, "M": cfg.M, "nnz": nnz, "hbm_peak_gbs": bw / 1e9, "fp64_peak_tflops": FP64_PEAK / 1e12,
           "rows": rows}
    if args.out:
        os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
        with open(args.out, "w") as f:
            json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
