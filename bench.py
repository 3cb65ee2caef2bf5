#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native ChFSI Chebyshev filter (Algorithm 1 step 1).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload si|al|tiny] [--impl reference]

One "step" = one whole pass of the hot path: one `ttdft_cheb_filter` call (all m fused recurrence
steps, all column panels) over one batch X of synthetic wavefunctions.  The default workload is
BASELINE.json's headline config 3 ("si": M=221,184, N=4,096, m=20).  Metric: useful fp64 GFLOP/s of
the filter = 2*nnz*N*m / t (nnz = non-zero entries of H; explicit zeros inside tiles earn nothing).

N > 1 (torchrun): column-band sharding (PAPER.md:L258 band parallelism with H replicated per
group): every rank filters its own N-column band with a full replica of H, no data-path
collective; "scaling": "weak".

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
column sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import synth  # noqa: E402

# fp64 ALU/DMMA peak derived from unit counts and clocks: 148 SMs x 64 fp64
# FMA/clk/SM x 2 flop x 1.965 GHz (clocks.max.sm).  Measured on this pool: DMMA loop 37.15 TFLOP/s.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# DRAM bytes per launch of the dominant kernel from ONE ncu --set full capture under profiles/
# (dram__bytes_read.sum + dram__bytes_write.sum), keyed by (workload, kernel): a number copied from that file, NOT measured
# in this run -- the line prints the file and the commit the capture was taken at beside it.  Missing key = not captured.
NCU_TRAFFIC = {("si", "bsr_i8"): (103.514e9 + 14.690e9, "profiles/r02_k3_si_full.txt", "5bdfe72"),
               ("si", "bsr_dmma"): (88.192e9 + 8.039e9, "profiles/r02_k1_si_full.txt", "228981b")}


def ncu_traffic(workload, kname):
    t = NCU_TRAFFIC.get((workload, kname))
    if t is None:
        return None, None
    return t[0], {"file": t[1], "commit": t[2], "note": "copied from that ncu --set full capture, not measured in this run"}
# nominal dense tensor-core ratio int8 : bf16 on B200 (4.5 : 2.25 Pop/s, B200_PROFILING.md table)
INT8_OVER_BF16 = 2.0


def int8_peak_tops():
    """Dense int8 tensor peak = measured bf16 peak (sustained: the kernel is timed inside a long step)
    x the nominal int8:bf16 ratio; falls back to the profiling guide's 1.4 PFLOP/s sustained figure."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            d = json.load(f)
        return INT8_OVER_BF16 * float(d["bf16_tflops_sustained"]), "of measured: MEASURED_PEAKS.json bf16_tflops_sustained x 2 (nominal int8:bf16)"
    except Exception:
        return INT8_OVER_BF16 * 1400.0, "of fallback: B200_PROFILING.md sustained bf16 1.4 PFLOP/s x 2 (nominal int8:bf16)"


def hbm_peak_gbs():
    """Measured HBM copy bandwidth (MEASURED_PEAKS.json), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured: MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "fallback: B200_PROFILING.md measured copy bandwidth 6.65 TB/s"


def load_bounds(name: str):
    with open(os.path.join(ROOT, "tests", "golden", "bounds.json")) as f:
        d = json.load(f)[name]
    return d["a"], d["b"], d["a0"]


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.power, self.reasons = [], [], set()
        self.sm_max = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop_evt.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join()
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "power_w_max": max(self.power),
                "samples": len(self.sm), "reasons": sorted(self.reasons)}


def gen_hamiltonian(cfg):
    H = synth.hamiltonian_bsr(cfg.G, cfg.b, cfg.z, cfg.seed)
    nnz = int(np.count_nonzero(H.values))
    return H, nnz


def oracle_sample_run(cfg, H, ncols_sample: int, m: int, bounds):
    """Time the oracle filter on `ncols_sample` seeded columns of the workload (exact: columns are independent)."""
    import oracle
    C = synth.bsr_to_csr_nonzeros(H)
    cols = synth.column_sample(cfg.N, cfg.panel, ncols_sample, cfg.seed)
    Xs = np.empty((cfg.M, len(cols)))
    for k, c in enumerate(cols):
        synth.dense_normal(cfg.M, 1, cfg.seed, synth.STREAM_X, col0=int(c), out=Xs[:, k:k + 1])
    a, b, a0 = bounds
    t0 = time.perf_counter()
    Y = oracle.cheb_filter(C.row_ptr, C.col_idx, C.values, Xs, m, a, b, a0)
    dt = time.perf_counter() - t0
    return dt, C.nnz, cols, Xs, Y, oracle.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, bounded sample, same metric and config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = synth.CONFIGS[args.workload]
    H, nnz = gen_hamiltonian(cfg)
    bounds = load_bounds(args.workload)
    ns = args.ref_cols
    import oracle
    oracle.lib()
    times = []
    for it in range(args.warmup + args.steps):
        dt, nnz_c, cols, _, _, threads = oracle_sample_run(cfg, H, ns, cfg.m, bounds)
        if it >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    gflops = 2.0 * nnz * len(cols) * cfg.m / t / 1e9
    sample = f"{len(cols)} seeded columns of {cfg.N} (all {cfg.M} rows, all m={cfg.m} steps) per step"
    line = {
        "impl": "reference", "metric": "ChFSI filter useful fp64 GFLOP/s", "value": gflops, "unit": "GFLOP/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, nnz, H.nblocks, args),
        "cpu_baseline": {"value": gflops, "unit": "GFLOP/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": gflops, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_sweep(sweep_argv):
    """Config 5 with parity: sweep.py times, the oracle checks each timed product on a seeded column sample."""
    import torch
    import oracle
    from paper_2110_15853_b200 import sweep

    def check(C, op, coeffs, X, Z, O):
        n = X.shape[1]
        cols = np.unique(np.concatenate([[0, n - 1], np.random.default_rng(n).integers(0, n, 14)]))
        cd = torch.from_numpy(cols).to(X.device)
        Xs, Zs, got = (np.ascontiguousarray(t[:, cd].cpu().numpy()) for t in (X, Z, O))
        if op == "spmm":
            ref = oracle.spmm(C.row_ptr, C.col_idx, C.values, coeffs[0], Xs)
        else:
            ref = oracle.cheb_step(C.row_ptr, C.col_idx, C.values, coeffs[0], coeffs[1], coeffs[2], Xs, Zs)
        return float(np.linalg.norm(got - ref) / np.linalg.norm(ref))

    sweep.main(sweep_argv, check=check)


def workload_config(cfg, nnz, nblocks, args):
    return {
        "workload": f"BASELINE.json config '{cfg.name}': G={cfg.G} b={cfg.b} M={cfg.M} N={cfg.N} m={cfg.m} "
                    f"z={cfg.z} (27-neighbour block-sparse symmetric H, seeded synthetic)",
        "M": cfg.M, "N": cfg.N, "m": cfg.m, "block": cfg.b, "nblocks": nblocks, "nnz": nnz,
        "panel_cols": args.panel if args.panel else cfg.panel,
        "l2": "inputs larger than L2 (H %.2f GB, X %.2f GB per rank)" % (nblocks * cfg.b * cfg.b * 8 / 1e9, cfg.M * cfg.N * 8 / 1e9),
        "parallelism": f"band x{args.gpus} (H replicated, columns sharded, no collective); "
                       + ("weak: every rank filters N columns" if getattr(args, "scaling", "weak") == "weak" else "strong: N columns cut into bands"),
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="si", choices=list(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--panel", type=int, default=0, help="column-panel width (0 = config default)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank filters its own N-column band (total work grows with N); strong = the config's N "
                         "columns are cut into N bands (e.g. --workload largest: 14,336 columns).  H is replicated either way.")
    ap.add_argument("--ref-cols", type=int, default=0,
                    help="columns in the oracle sample; 0 = 48 for the cpu_baseline leg (about 18 s on 16 host cores) and 16 per step "
                         "for --impl reference (about 6 s per step, so that any --steps/--warmup ends within a few minutes)")
    ap.add_argument("--math", default="auto", choices=["auto", "fp64", "i8", "i8x7"],
                    help="arithmetic of the block product: fp64 DMMA; exact int8 digit planes on the tcgen05 tensor "
                         "cores with 7 planes (55 bits, i8x7) or 6 planes (47 bits, i8); auto = i8x7 for tiles >= 64")
    ap.add_argument("--no-other-modes", action="store_true", help="skip the short runs of the other math modes")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-project", action="store_true", help="skip the subspace-projection (NEXT-1) measurement")
    ap.add_argument("--sweep", nargs=argparse.REMAINDER, default=None,
                    help="BASELINE.json config 5 instead of the headline: the timings of paper_2110_15853_b200.sweep (its own options may "
                         "follow, e.g. --sweep --ns 16,256 --layouts bsr,csr) with a relerr column -- every timed product compared with "
                         "the CPU oracle on 16 seeded columns (columns are independent in one product)")
    args = ap.parse_args()
    if args.sweep is not None:
        return run_sweep(args.sweep)
    if args.ref_cols <= 0:
        args.ref_cols = 16 if args.impl == "reference" else 48
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2110_15853_b200 as tt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = synth.CONFIGS[args.workload]
    a, b, a0 = load_bounds(args.workload)
    H, nnz = gen_hamiltonian(cfg)
    dev = torch.device("cuda", local)
    t_up0 = time.perf_counter()
    h_dev = (torch.from_numpy(H.row_ptr).to(dev), torch.from_numpy(H.col_idx).to(dev), torch.from_numpy(H.values).to(dev))
    torch.cuda.synchronize()
    t_upload = time.perf_counter() - t_up0                   # pageable host -> device copy of the input arrays (not the library)
    t_build0 = time.perf_counter()
    Hd = tt.h_build_bsr(H.M, H.b, *h_dev, flags=tt.CHECK_SORTED | tt.CHECK_SYMMETRY)     # A0: checks, format, digit planes
    torch.cuda.synchronize()
    t_build = time.perf_counter() - t_build0
    del h_dev
    MODES = {"auto": tt.MATH_AUTO, "fp64": tt.MATH_FP64, "i8": tt.MATH_I8, "i8x7": tt.MATH_I8X7}
    Hd.set_math_mode(MODES[args.math])
    info = Hd.info()
    assert info["kernel"] == 1, "a block-sparse tensor-core kernel must be the one that runs"
    use_i8 = info["math"] in (tt.MATH_I8, tt.MATH_I8X7)
    planes = {tt.MATH_I8: 6, tt.MATH_I8X7: 7}.get(info["math"], 0)
    mode_name = {tt.MATH_FP64: "fp64", tt.MATH_I8: "i8", tt.MATH_I8X7: "i8x7"}[info["math"]]

    # this rank's band of wavefunctions (host, pinned).  weak: columns [rank*N, (rank+1)*N) of a global block of world*N columns;
    # strong: the config's own N columns cut into `world` bands (PAPER.md:L258 band parallelism, paper's partition rule L244-248)
    from paper_2110_15853_b200 import bands
    if args.scaling == "strong":
        band0, ncols = bands.band_of(rank, world, cfg.N)
        total_cols = cfg.N
    else:
        band0, ncols = bands.weak_band(rank, cfg.N)
        total_cols = cfg.N * world
    Xh = torch.empty((cfg.M, ncols), dtype=torch.float64).pin_memory()
    synth.dense_normal(cfg.M, ncols, cfg.seed, synth.STREAM_X, col0=band0, out=Xh.numpy())
    Yh = torch.empty((cfg.M, ncols), dtype=torch.float64).pin_memory()
    Xd = Xh.to(dev, non_blocking=True)
    Yd = torch.empty_like(Xd)
    panel = args.panel if args.panel else cfg.panel
    torch.cuda.synchronize()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    npanels = -(-ncols // (panel if panel else min(ncols, 4096)))
    useful = 2.0 * nnz * ncols * cfg.m                                   # flops of the method: non-zeros of H only
    executed = 2.0 * H.nblocks * cfg.b * cfg.b * ncols * cfg.m           # what dense tiles multiply (explicit zeros included)
    alg_bytes = cfg.m * (npanels * 8.0 * nnz + 24.0 * cfg.M * ncols) - 8.0 * cfg.M * ncols
    hbm_bw, hbm_src = hbm_peak_gbs()
    t_roof = max(alg_bytes / (hbm_bw * 1e9), useful / (FP64_PEAK_TFLOPS * 1e12))   # SURVEY.md 8(d) (iv), whole filter
    binds = "fp64" if useful / (FP64_PEAK_TFLOPS * 1e12) >= alg_bytes / (hbm_bw * 1e9) else "hbm"

    def timed_filter(mode):
        """W warm-up + K timed ttdft_cheb_filter calls in one math mode: device time (max over ranks), the library's own CUDA
        event pairs per kernel, clocks sampled during the timed region, kernel launches counted by the library."""
        Hd.set_math_mode(mode)
        work = torch.empty(tt.cheb_filter_work_bytes(Hd, ncols, panel) + 16, dtype=torch.uint8, device=dev)

        def step():
            tt.cheb_filter(Hd, Xd, Yd, cfg.m, a, b, a0, panel_cols=panel, work=work)

        for _ in range(args.warmup):
            step()
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        for k in tt.KERNEL_IDS:
            tt.timing_read(k)
        tt.timing_enable(True)       # CUDA event pairs around every library kernel, on the launching stream
        n0 = tt.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            step()
        e1.record()
        barrier()
        launches = tt.launch_count() - n0
        tt.timing_enable(False)
        ktimes = {k: tt.timing_read(k) for k in tt.KERNEL_IDS}
        clocks = sampler.stop()
        t_region = e0.elapsed_time(e1) * 1e-3
        if dist is not None:
            tmax = torch.tensor([t_region], dtype=torch.float64, device=dev)
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
            t_region = float(tmax.item())
        del work
        return {"t_step": t_region / args.steps, "t_region": t_region, "ktimes": ktimes, "clocks": clocks, "launches": int(launches)}

    def mode_report(run, use_i8, planes):
        """roofline object of one timed run (dominant kernel = the fused step kernel; one launch = one recurrence step over one panel;
        its launch time comes from the library's CUDA event pairs recorded inside the timed region)."""
        kname = "bsr_i8" if use_i8 else "bsr_dmma"
        k_ms, k_n = run["ktimes"][kname]
        assert k_n == args.steps * cfg.m * npanels, (k_n, args.steps, cfg.m, npanels)
        t_launch = k_ms * 1e-3 / k_n
        nl = cfg.m * npanels
        shares = {k: v[0] / (run["t_region"] * 1e3) for k, v in run["ktimes"].items() if v[1]}
        traffic, traffic_src = ncu_traffic(args.workload, kname)
        common = {"launch_ms": t_launch * 1e3, "step_share": shares, "traffic": traffic, "traffic_source": traffic_src,
                  "hbm_alg_gbs": alg_bytes / run["t_step"] / 1e9,
                  # T_roof / t for the WHOLE filter, T_roof = max(alg. bytes / HBM peak, useful flops / fp64 peak)
                  "survey_frac": t_roof / run["t_step"], "survey_binds": binds,
                  "survey_t_roof_ms": t_roof * 1e3, "survey_peaks": {"fp64_tflops": FP64_PEAK_TFLOPS, "hbm_gbs": hbm_bw, "hbm_source": hbm_src}}
        if use_i8:
            # K3: the product runs as S(S+1)/2 exact int8 digit-plane products on the tensor pipe, so the tensor pipe bounds it.
            # Algorithmic ops per launch = 2 * pairs * nnz * N (non-zeros only); executed = dense tiles, padded to the MMA shape.
            pairs = planes * (planes + 1) // 2
            peak, peak_src = int8_peak_tops()
            ops_launch = 2.0 * pairs * nnz * ncols / npanels
            mrows = cfg.b if cfg.b in (64, 96) else 128        # K3T (the default for 64- and 96-wide tiles) multiplies no padding rows
            ops_exec = 2.0 * pairs * H.nblocks * mrows * cfg.b * (-(-ncols // 64) * 64) / npanels
            roof = {"bound": "tensor", "achieved": ops_launch / t_launch / 1e12, "peak": peak, "unit": "TFLOP/s",
                    "frac": ops_launch / t_launch / 1e12 / peak, "kernel": "ttdft::bsr_i8_kernel", "peak_source": peak_src,
                    "ops": f"int8 multiply-add = 2 ops; {pairs} digit-plane products per fp64 product ({planes} planes per operand: "
                           "the implementation's choice of arithmetic, not the method's work)",
                    "executed_tops": ops_exec / t_launch / 1e12, "executed_frac": ops_exec / t_launch / 1e12 / peak,
                    # the measured-peak figure above is 2 x a power-limited cuBLAS bf16 rate, which an int8 kernel can exceed
                    # (fewer joules per op): the nominal dense 8-bit peak (B200_PROFILING.md's fp8 row, 4.5 Pop/s; int8 has the same rate) is the hard ceiling
                    "peak_nominal": 4500.0, "executed_frac_of_nominal": ops_exec / t_launch / 1e12 / 4500.0,
                    "dense_tile_ceiling": useful / executed,
                    "useful_fp64_tflops_kernel": useful / nl / t_launch / 1e12}
        else:
            ach = useful / nl / t_launch / 1e12
            roof = {"bound": "alu", "achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach / FP64_PEAK_TFLOPS,
                    "kernel": "ttdft::bsr_dmma_kernel",
                    "peak_source": "derived: 148 SM x 64 fp64 FMA/clk x 2 x 1.965 GHz (native fp64 ALU/DMMA pipe; fp64 has no entry in "
                                   "MEASURED_PEAKS.json)",
                    "executed_tflops": executed / nl / t_launch / 1e12, "executed_frac": executed / nl / t_launch / 1e12 / FP64_PEAK_TFLOPS,
                    "dense_tile_ceiling": useful / executed}
        roof.update(common)
        return roof

    DTYPE = {"fp64": "f64 (fp64 tensor-core MMA, fp64 accumulate)",
             "i8x7": "f64 in/out; int8x7 digit planes (55 bits below each row/column maximum), exact int32 accumulate, fp64 recombine",
             "i8": "f64 in/out; int8x6 digit planes (47 bits below each row/column maximum), exact int32 accumulate, fp64 recombine"}

    run = timed_filter(MODES[args.math])
    t_step, clocks = run["t_step"], run["clocks"]
    roof = mode_report(run, use_i8, planes)
    try:
        roof["peak_measured_dmma"] = tt.probe_fp64_peak(1, 300)
    except Exception:
        pass
    cols_d = torch.from_numpy(synth.column_sample(ncols, cfg.panel, args.ref_cols, cfg.seed)).to(dev)
    samples = {mode_name: Yd[:, cols_d].clone()}
    Yd_headline = None                          # kept for the e2e leg's bit-for-bit check, if it fits beside X, Y and the scratch
    if not args.no_e2e and torch.cuda.mem_get_info(dev)[0] > 2 * Yd.numel() * 8:
        Yd_headline = Yd.clone()

    line = {
        "metric": "ChFSI filter useful fp64 GFLOP/s", "value": 2.0 * nnz * total_cols * cfg.m / t_step / 1e9, "unit": "GFLOP/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_step * 1e3,
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": DTYPE[mode_name], "data": "synthetic",
        "config": workload_config(cfg, nnz, H.nblocks, args),      # the same object the reference arm prints
        "math": (f"{mode_name}: exact int8 digit planes on tcgen05 ({planes} x 8 bit per fp64 operand = "
                 f"{8 * planes - 1} bits below the row/column maximum, exact int32 accumulation, fp64 "
                 "recombination, fp64 in/out)") if use_i8 else "fp64: fp64 tensor-core MMA (DMMA)",
        "clocks": clocks, "gpu_launches": run["launches"], "roofline": roof,
        "h_build_ms": t_build * 1e3, "h_upload_ms": t_upload * 1e3,
    }

    # ---- the native-fp64 arithmetic (TTDFT_MATH_FP64, kernel K1) with EQUAL standing: same handle, inputs, --steps and --warmup ----
    others = {}
    if not args.no_other_modes and mode_name != "fp64":
        r64 = timed_filter(MODES["fp64"])
        samples["fp64"] = Yd[:, cols_d].clone()
        line["fp64_native"] = {
            "what": "the same filter in TTDFT_MATH_FP64: every product on the fp64 tensor-core pipe (DMMA), no digit planes",
            "metric": line["metric"], "value": 2.0 * nnz * total_cols * cfg.m / r64["t_step"] / 1e9, "unit": "GFLOP/s", "dtype": DTYPE["fp64"],
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r64["t_step"] * 1e3, "clocks": r64["clocks"],
            "gpu_launches": r64["launches"], "roofline": mode_report(r64, False, 0)}
        others["fp64"] = line["fp64_native"]

    # ---- end to end through the C-ABI host-buffer call: H2D of X and D2H of Y inside the timed region
    if not args.no_e2e:
        Hd.set_math_mode(MODES[args.math])
        # default panel schedule (a ramp up to 2,048 columns) if its scratch fits beside the resident X and Y, else uniform 1,024 / 512
        hp = 0
        for hp in (0, 1024, 512):
            if tt.cheb_filter_host_work_bytes(Hd, ncols, hp) + (2 << 30) < torch.cuda.mem_get_info(dev)[0]:
                break
        hwork = torch.empty(tt.cheb_filter_host_work_bytes(Hd, ncols, hp) + 1024, dtype=torch.uint8, device=dev)
        tt.cheb_filter_host(Hd, Xh, Yh, cfg.m, a, b, a0, panel_cols=hp, work=hwork)   # warm-up
        barrier()
        t0 = time.perf_counter()
        nrep = max(1, min(args.steps, 2))
        for _ in range(nrep):
            tt.cheb_filter_host(Hd, Xh, Yh, cfg.m, a, b, a0, panel_cols=hp, work=hwork)
        barrier()
        t_e2e = (time.perf_counter() - t0) / nrep
        if dist is not None:
            tm = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
            dist.all_reduce(tm, op=dist.ReduceOp.MAX)
            t_e2e = float(tm.item())
        line["e2e"] = {"value": 2.0 * nnz * total_cols * cfg.m / t_e2e / 1e9, "unit": "GFLOP/s",
                       "h2d_bytes_per_step": cfg.M * ncols * 8, "d2h_bytes_per_step": cfg.M * ncols * 8,
                       "ms_per_step": t_e2e * 1e3, "api": "ttdft_cheb_filter_host (pinned host X, Y; " + ("default panel schedule: 256 | 768 | 2048 ... | 768 | 256 columns)" if hp == 0
                                                                              else f"{hp}-column panels: the default schedule's scratch does not fit beside the resident X, Y)"),
                       # sanity: the host path and the device path agree bit for bit on this rank's band
                       "matches_device_path": None}
        del hwork
        if Yd_headline is not None:             # compared in column chunks: no second full copy on the device
            same = True
            for c0 in range(0, ncols, 1024):
                same = same and bool(torch.equal(Yh[:, c0:c0 + 1024].to(dev), Yd_headline[:, c0:c0 + 1024]))
            line["e2e"]["matches_device_path"] = same
        del Yd_headline

    # ---- the 6-plane int8 mode on the same handle and inputs: 1 warm-up + 1 timed filter ----
    if rank == 0 and world == 1 and not args.no_other_modes:
        for name in ("i8x7", "i8"):
            if name == mode_name or not info["i8_planes"]:
                continue
            Hd.set_math_mode(MODES[name])
            w2 = torch.empty(tt.cheb_filter_work_bytes(Hd, ncols, panel) + 16, dtype=torch.uint8, device=dev)
            tt.cheb_filter(Hd, Xd, Yd, cfg.m, a, b, a0, panel_cols=panel, work=w2)
            torch.cuda.synchronize()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record()
            tt.cheb_filter(Hd, Xd, Yd, cfg.m, a, b, a0, panel_cols=panel, work=w2)
            f1.record()
            torch.cuda.synchronize()
            t_o = f0.elapsed_time(f1) * 1e-3
            others[name] = {"value": useful / t_o / 1e9, "unit": "GFLOP/s", "dtype": DTYPE[name], "ms_per_step": t_o * 1e3,
                            "steps": 1, "warmup": 1, "survey_frac": t_roof / t_o}
            samples[name] = Yd[:, cols_d].clone()
            del w2
        line["other_math_modes"] = {k: v for k, v in others.items() if k != "fp64"}
    Hd.set_math_mode(MODES[args.math])

    # ---- NEXT-1: subspace projection H_F = X^T (H X) on the same handle and X (1 warm-up + 2 timed) ----
    if rank == 0 and world == 1 and not args.no_project:
        Gd = torch.empty((cfg.N, cfg.N), dtype=torch.float64, device=dev)
        pw = torch.empty(tt.project_work_bytes(Hd, cfg.N) + 1024, dtype=torch.uint8, device=dev)
        tt.project(Hd, Xd, Gd, work=pw)
        torch.cuda.synchronize()
        for k in tt.KERNEL_IDS:
            tt.timing_read(k)
        tt.timing_enable(True)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for _ in range(2):
            tt.project(Hd, Xd, Gd, work=pw)
        g1.record()
        torch.cuda.synchronize()
        tt.timing_enable(False)
        pk = {k: tt.timing_read(k) for k in tt.KERNEL_IDS}
        t_p = g0.elapsed_time(g1) * 1e-3 / 2
        gram_ms = pk["gram_i8"][0] / 2                 # K4's time per ttdft_project call (the product runs as several launches)
        gram_launches = pk["gram_i8"][1] // 2
        # The handle was built with TTDFT_CHECK_SYMMETRY, so H_F = H_F^T is known and ttdft_project computes only the entries on and
        # above the diagonal (the method's own work: N(N+1)/2 entries of 2M flops), as whole 128 x 128 tile groups (executed work).
        n128 = -(-cfg.N // 128)
        fl_gram = 2.0 * cfg.M * cfg.N * (cfg.N + 1) / 2
        fl_gram_exec = 2.0 * (-(-cfg.M // 128) * 128) * 128 * 128 * n128 * (n128 + 1) / 2
        fl_gram_dense = 2.0 * cfg.M * cfg.N * cfg.N
        fl_spmm = 2.0 * nnz * cfg.N
        peak8, peak8_src = int8_peak_tops()
        line["project"] = {
            "what": "H_F = X^T (H X), Algorithm 1 step 3 (ttdft_project): one K3 step + Gram product K4 on the int8 tensor cores; "
                    "H = H^T was verified at build, so only the upper triangle of H_F is computed and mirrored",
            "ms": t_p * 1e3, "useful_fp64_tflops": (fl_gram + fl_spmm) / t_p / 1e12, "steps": 2, "warmup": 1,
            "kernels_ms_each": {k: v[0] / v[1] for k, v in pk.items() if v[1]},
            "gram_roofline": {"bound": "tensor", "achieved": 28.0 * fl_gram / (gram_ms * 1e-3) / 1e12, "peak": peak8, "unit": "TFLOP/s",
                              "frac": 28.0 * fl_gram / (gram_ms * 1e-3) / 1e12 / peak8, "peak_source": peak8_src, "launch_ms": gram_ms,
                              "launches": gram_launches,       # launch_ms is their sum: the whole Gram product
                              "ops": "method's own work: N(N+1)/2 entries x 2M flops x 28 digit-plane products",
                              "executed_tops": 28.0 * fl_gram_exec / (gram_ms * 1e-3) / 1e12,
                              "executed_frac": 28.0 * fl_gram_exec / (gram_ms * 1e-3) / 1e12 / peak8,
                              "useful_fp64_tflops": fl_gram / (gram_ms * 1e-3) / 1e12,
                              "dense_equivalent_fp64_tflops": fl_gram_dense / (gram_ms * 1e-3) / 1e12},
            "symmetry_defect": float(((Gd - Gd.T).norm() / Gd.norm()).item()),
        }
        if not args.no_cpu_baseline:
            # oracle on a seeded sub-block: G[cols, cols] = X_c^T (H X_c) (entry (j,l) depends on columns j and l only)
            import oracle
            pc = synth.column_sample(cfg.N, cfg.panel, args.ref_cols, cfg.seed)
            Cn = synth.bsr_to_csr_nonzeros(H)
            Xc = np.ascontiguousarray(Xd[:, torch.from_numpy(pc).to(dev)].cpu().numpy())
            ref = oracle.project(Cn.row_ptr, Cn.col_idx, Cn.values, Xc)
            gotp = Gd[torch.from_numpy(pc).to(dev)][:, torch.from_numpy(pc).to(dev)].cpu().numpy()
            line["project"]["gpu_vs_oracle_relerr_on_sample"] = float(np.linalg.norm(gotp - ref) / np.linalg.norm(ref))
            del Cn
        del Gd, pw
        # ---- Algorithm 1 step 5: rotation Psi = X Q (ttdft_rotate), Q a seeded N x N matrix (1 warm-up + 2 timed) ----
        Qd = torch.randn(cfg.N, cfg.N, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(cfg.seed))
        rw = torch.empty(tt.rotate_work_bytes(cfg.M, cfg.N, cfg.N) + 1024, dtype=torch.uint8, device=dev)
        tt.rotate(Xd, Qd, Yd, work=rw)
        torch.cuda.synchronize()
        g0.record()
        for _ in range(2):
            tt.rotate(Xd, Qd, Yd, work=rw)
        g1.record()
        torch.cuda.synchronize()
        t_r = g0.elapsed_time(g1) * 1e-3 / 2
        ops_rot = 28.0 * fl_gram_dense                     # Q is a full matrix here: every entry of the product is the method's work
        line["rotate"] = {"what": "Psi = X Q, Algorithm 1 step 5 (ttdft_rotate): kernel K3 on row-scaled digit tiles of X (Q dense)",
                          "ms": t_r * 1e3, "useful_fp64_tflops": fl_gram_dense / t_r / 1e12, "steps": 2, "warmup": 1,
                          "int8_tops": ops_rot / t_r / 1e12, "frac_of_int8_peak": ops_rot / t_r / 1e12 / peak8}
        if not args.no_cpu_baseline:
            rr = torch.from_numpy(np.unique(np.random.default_rng(cfg.seed).integers(0, cfg.M, 16))).to(dev)
            refr = oracle.rotate(np.ascontiguousarray(Xd[rr].cpu().numpy()), Qd.cpu().numpy())
            line["rotate"]["gpu_vs_oracle_relerr_on_sample"] = float(np.linalg.norm(Yd[rr].cpu().numpy() - refr) / np.linalg.norm(refr))
        del Qd, rw
        # ---- Algorithm 1 step 2: X_F = Orth(X) (ttdft_orthonormalize, Cholesky-QR2; 1 warm-up + 1 timed) ----
        ow = torch.empty(tt.orthonormalize_work_bytes(cfg.M, cfg.N, 2) + 1024, dtype=torch.uint8, device=dev)
        tt.orthonormalize(Xd, Yd, passes=2, work=ow)
        torch.cuda.synchronize()
        g0.record()
        tt.orthonormalize(Xd, Yd, passes=2, work=ow)
        g1.record()
        torch.cuda.synchronize()
        t_o = g0.elapsed_time(g1) * 1e-3
        # method's own work of Cholesky-QR2: per pass N(N+1)/2 entries of X^T X and the triangular product X R^-1 (M N(N+1)/2
        # multiply-adds each), plus the n x n Cholesky and triangular inverse (n^3/3 flops each)
        fl_orth = 2 * (2 * fl_gram + 2.0 * cfg.N ** 3 / 3)
        line["orthonormalize"] = {"what": "X_F = Orth(X), Algorithm 1 step 2 (ttdft_orthonormalize): Cholesky-QR2 = 2 x (Gram product K4 on the "
                                          "upper triangle, n x n Cholesky + inverse, triangular rotation X R^-1 on K3)",
                                  "ms": t_o * 1e3, "useful_fp64_tflops": fl_orth / t_o / 1e12, "steps": 1, "warmup": 1,
                                  "dense_equivalent_fp64_tflops": 8.0 * cfg.M * cfg.N * cfg.N / t_o / 1e12}
        if not args.no_cpu_baseline:
            lead = 16      # column j of Q depends on columns 0..j of X only: the leading block against the oracle's Gram-Schmidt
            refq = oracle.orthonormalize(np.ascontiguousarray(Xd[:, :lead].cpu().numpy()))
            line["orthonormalize"]["gpu_vs_oracle_relerr_on_sample"] = float(np.linalg.norm(Yd[:, :lead].cpu().numpy() - refq) / np.linalg.norm(refq))
        del ow

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        dt, _, cols, Xs, Yo, threads = oracle_sample_run(cfg, H, args.ref_cols, cfg.m, (a, b, a0))
        got = samples[mode_name].cpu().numpy()
        err = float(np.linalg.norm(got - Yo) / np.linalg.norm(Yo))
        for name in others:
            g2 = samples[name].cpu().numpy()
            others[name]["gpu_vs_oracle_relerr_on_sample"] = float(np.linalg.norm(g2 - Yo) / np.linalg.norm(Yo))
        line["cpu_baseline"] = {"value": 2.0 * nnz * len(cols) * cfg.m / dt / 1e9, "unit": "GFLOP/s", "cores": threads,
                                "kind": "oracle", "seconds": dt,
                                "sample": f"{len(cols)} seeded columns of {cfg.N} (all rows, all m={cfg.m} steps)",
                                "gpu_vs_oracle_relerr_on_sample": err}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
