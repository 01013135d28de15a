#!/usr/bin/env python
"""bench.py -- Chebyshev-filter throughput on B200 (BASELINE.json metric).

A "step" is one chase_filter_ws call (the whole hot path: host scalars + schedule, one fused
TMA/DMMA step kernel per degree) on the workload BASELINE.json quotes the metric on:
cfg 4 = N=40000 complex128 GUE, V0 40000x2000, sorted even degrees 8..36 (synthetic, seeded).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

Prints ONE JSON line (rank 0).  `value` = filter GFLOP/s = 8 N^2 sum(deg) / t (complex; 2 N^2
sum(deg) real), whole job, inputs resident in HBM.  `e2e` = same metric through
chase_filter_host (HOST buffers, H2D/D2H inside the timed region).  `roofline` = achieved
TFLOP/s of the step kernel vs the FP64 peak.  `cpu_baseline` = the oracle,
as it stands, on the host cores on a bounded sample.  `parity` = the timed run's result against the
oracle on the SURVEY 8(c) column sample (>= 32 columns, own degrees, full H).  `all_configs` = the other
BASELINE.json configs (1, 2, 3, 5), each timed the same way with its own clock record, roofline
fraction and oracle comparison.  --impl reference times the oracle.
Multi-GPU (--gpus N under torchrun): independent column batches per rank, H replicated, no
data-path collective; scaling = weak.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from paper_1805_10121_b200 import workloads as W

METRIC = "chebyshev_filter_gflops"
UNIT = "GFLOP/s"
# FP64 peak: 148 SMs x 128 FP64 flop/clk/SM x 1.965 GHz (clocks.max.sm).
# The DMMA.8x8x4 and DFMA pipes have the same rate; a register-only probe run live below
# (chase_fp64_peak_probe) measures it on this very GPU.
FP64_FLOP_PER_CLK_SM = 128
TF32_OVER_BF16_NOMINAL = 1.1 / 2.25      # B200_PROFILING.md nominal dense peaks: tf32 1.1, bf16 2.25 PFLOP/s


# dram__bytes_read.sum + dram__bytes_write.sum of one full-width step launch (ncu --set full captures).
# NOT measured in this run: typed in from the committed capture named in each note.
NCU_TRAFFIC = {
    4: (157.315675e9 + 1.352249e9, "bytes of one full-width launch (2000 columns; algorithmic 30.7e9; 145-157e9 over three "
                                   "captures); from profiles/ncu_r2_step_dmma.md, not measured in this run"),
    5: (134.158879e9 + 1.454750e9, "bytes of one full-width launch (3000 columns; algorithmic 28.8e9 + vectors); "
                                   "from profiles/ncu_r2_step_tf32.md, not measured in this run"),
    3: (9.788422e9 + 0.232516e9, "bytes of one full-width launch (1400 columns; algorithmic 3.2e9 + 0.45e9 of vectors); "
                                 "from profiles/ncu_r3_step_dmma_f64.md, not measured in this run"),
    2: (328.881152e6 + 18.007808e6, "bytes of one full-width launch (256 columns; algorithmic 268e6 + vectors); "
                                    "from profiles/ncu_r2_step_dmma.md, not measured in this run"),
}


def measured_bf16_sustained_tflops():
    """(TFLOP/s, source): the driver-written sustained bf16 GEMM rate (the step kernel is timed inside a
    long step), else the nominal dense figure."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            m = json.load(f)
        return float(m["bf16_tflops_sustained"]), "MEASURED_PEAKS.json bf16_tflops_sustained"
    except (OSError, KeyError, ValueError):
        return 2250.0, "nominal bf16 dense 2250 TFLOP/s (MEASURED_PEAKS.json absent)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based); 4 = metric config")
    ap.add_argument("--N", type=int, default=None, help="override N (debug only; prints config.reduced)")
    ap.add_argument("--ncols", type=int, default=None)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-aux", action="store_true", help="skip the hemm / residuals / Lanczos timings")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the cfg 1/2/3/5 block of the JSON line")
    ap.add_argument("--sample-cols", type=int, default=16)
    ap.add_argument("--sample-degree", type=int, default=8)
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            t0 = time.perf_counter()          # short timed regions: make sure the sampler is already running
            while not self.lines and time.perf_counter() - t0 < 3.0:
                time.sleep(0.02)
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_setup(ngpus: int):
    """(rank, world, local_rank); initialises NCCL only when launched under torchrun."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local))
    return rank, world, local


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


def max_over_ranks(x: float, world: int) -> float:
    if world == 1:
        return x
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world: int) -> float:
    if world == 1:
        return x
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------------------------
# workload
# ----------------------------------------------------------------------------------------------
def build_workload(args, device, rank: int) -> W.Workload:
    w = W.make_config(args.config, device=device, N=args.N, ncols=args.ncols)
    if rank > 0:   # independent batch per rank: same H (replicated), different seeded V0
        seed = W.BASE_SEED + 1000 * args.config + 1 + 10 * rank
        w.V0 = W.gaussian_colmajor(w.N, w.ncols, w.dtype, seed, device)
    return w


def workload_config(args, w: W.Workload, world: int) -> dict:
    cfg = {
        "workload": f"BASELINE.json configs[{args.config - 1}] (cfg {args.config}): N={w.N} "
                    f"{W.DTYPE_NAMES[w.dtype]} Hermitian, V0 {w.N}x{w.ncols}, degrees "
                    f"{int(w.degrees.min())}..{int(w.degrees.max())} sorted, sum_deg={w.sum_deg}",
        "N": w.N, "ncols_per_gpu": w.ncols, "sum_deg_per_gpu": w.sum_deg,
        "a": w.a, "b": w.b, "lambda1": w.lambda1,
        "l2": (f"inputs exceed L2 (H = {w.H.numel() * w.H.element_size() / 1e9:.1f} GB > 126 MB); no flush needed"
               if w.H.numel() * w.H.element_size() >= (512 << 20) else "L2 flushed (512 MB write) between iterations"),
        "parallelism": "single GPU" if world == 1 else f"{world} independent column batches, H replicated, no collective",
    }
    if args.N is not None or args.ncols is not None:
        cfg["reduced"] = True
    return cfg


def sample_columns(w: W.Workload, k: int):
    k = min(k, w.ncols)
    return [int(round(i * (w.ncols - 1) / max(k - 1, 1))) for i in range(k)] if k > 1 else [0]


def host_colmajor_numpy(x: torch.Tensor) -> np.ndarray:
    """Device (or host) column-major tensor -> Fortran-ordered numpy array, one copy."""
    return x.t().cpu().t().numpy()


def oracle_sample_run(Hn: np.ndarray, Vn: np.ndarray, degree: int, w):
    """Times the oracle, as it stands, on `Vn` (column sample) with a uniform truncated degree.
    Returns (seconds, flops, result)."""
    import oracle
    deg = np.full(Vn.shape[1], degree, dtype=np.int32)
    f = 8.0 if np.iscomplexobj(Hn) else 2.0
    t0 = time.perf_counter()
    out = oracle.chase_filter(Hn, Vn, deg, w.a, w.b, w.lambda1)
    dt = time.perf_counter() - t0
    return dt, f * float(Hn.shape[0]) ** 2 * Vn.shape[1] * degree, out


def time_aux_ops(pkg, w, Y, device):
    """Device times of chase_hemm (Rayleigh-Ritz A Q^, all columns), chase_residuals and chase_lanczos
    (k = 25, 1 + 4 runs; Table 1 defaults) on the bench workload.  One warm-up, one timed call each."""
    N, n, dtype = w.N, w.ncols, w.dtype
    f = 8.0 if dtype.is_complex else 2.0

    def timed(fn):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    out = {}
    ms = timed(lambda: pkg.chase_hemm(w.H, w.V0, Y))
    out["chase_hemm"] = {"ms": ms, "gflops": f * N * N * n / ms * 1e-6, "ncols": n}
    ritz = np.linspace(w.lambda1, w.a, n)
    rws = torch.empty(pkg.chase_residuals_workspace_bytes(N, n, dtype), dtype=torch.uint8, device=device)
    ms = timed(lambda: pkg.chase_residuals(w.H, w.V0, ritz, workspace=rws))
    out["chase_residuals"] = {"ms": ms, "gflops": f * N * N * n / ms * 1e-6, "ncols": n}
    del rws
    k, nruns = 25, 5
    lws = torch.empty(pkg.chase_lanczos_workspace_bytes(N, nruns, k, dtype), dtype=torch.uint8, device=device)
    V0 = W.as_colmajor(w.V0[:, :nruns])
    res = {}
    ms = timed(lambda: res.update(ab=pkg.chase_lanczos(w.H, V0, k, workspace=lws)))
    b_sup, mu1, mune = pkg.chase_spectral_estimates(res["ab"][0], res["ab"][1], N, n)
    h_bytes = N * N * w.H.element_size()
    out["chase_lanczos"] = {"ms": ms, "k": k, "runs": nruns, "hbm_gbs_over_H": k * h_bytes / ms * 1e-6,
                            "b_sup": b_sup, "mu_1": mu1, "mu_nev_nex": mune}
    return out


# ----------------------------------------------------------------------------------------------
# --impl reference : the oracle on the host cores (tier framing (4))
# ----------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    device = torch.device("cuda:0") if torch.cuda.is_available() else torch.device("cpu")
    w = build_workload(args, device, 0)    # the GPU, if present, only generates the inputs
    cols = sample_columns(w, args.sample_cols)
    Hn = host_colmajor_numpy(w.H)
    Vn = np.asfortranarray(host_colmajor_numpy(w.V0)[:, cols])
    cfg = workload_config(args, w, 1)
    N, ncols = w.N, w.ncols
    w.H = None
    w.V0 = None
    if device.type == "cuda":
        torch.cuda.empty_cache()
    for _ in range(args.warmup):
        oracle_sample_run(Hn, Vn, args.sample_degree, w)
    times, flops = [], 0.0
    for _ in range(args.steps):
        dt, fl, _ = oracle_sample_run(Hn, Vn, args.sample_degree, w)
        times.append(dt)
        flops = fl
    total = sum(times)
    value = flops * args.steps / total * 1e-9
    sample = (f"{len(cols)} of {ncols} columns (evenly spaced), full {N}x{N} H, degree truncated to "
              f"{args.sample_degree}; one step = one oracle call on that sample")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": cfg,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "nproc": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
DTYPE_LABEL = {torch.complex128: "c128 (f64 arithmetic)", torch.float64: "f64",
               torch.complex64: "c64 (f32 arithmetic)", torch.float32: "f32"}


def time_filter(pkg, w, steps: int, warmup: int, device, world: int, rank: int, local: int):
    """W untimed + K timed chase_filter_ws calls on workload `w` (V restored from V0 and, for inputs
    that fit in L2, the L2 flushed outside the timed region; CUDA events on the launching stream;
    nvidia-smi clocks sampled during the timed region).  Returns a dict; `dev_s` is this rank's."""
    N, n, dtype = w.N, w.ncols, w.dtype
    V = W.empty_colmajor(N, n, dtype, device)
    ws = torch.empty(pkg.chase_filter_workspace_bytes(N, n, dtype), dtype=torch.uint8, device=device)
    stream = torch.cuda.Stream(device)
    h_bytes = w.H.numel() * w.H.element_size()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device) if h_bytes < (512 << 20) else None

    def one_step(timed: bool):
        V.copy_(w.V0)                       # restore V0 outside the timed region
        if flush is not None:
            flush.zero_()                   # inputs fit in L2: flush it between iterations
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            pkg.chase_filter_ws(w.H, V, w.degrees, w.a, w.b, w.lambda1, ws, stream=stream)
            e1.record(stream)
        torch.cuda.current_stream().wait_stream(stream)
        return (e0, e1) if timed else None

    for _ in range(warmup):
        one_step(False)
    barrier(world)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = pkg.chase_filter_launch_count()
    barrier(world)
    t_wall0 = time.perf_counter()
    events = [one_step(True) for _ in range(steps)]
    barrier(world)
    t_wall = time.perf_counter() - t_wall0
    launches = pkg.chase_filter_launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms = [e0.elapsed_time(e1) for e0, e1 in events]
    return {"dev_s": sum(ms) * 1e-3, "ms": ms, "launches": launches, "clocks": clocks, "t_wall": t_wall, "V": V}


def roofline_of(pkg, w, achieved_tflops: float, clocks, device, launches_per_step: int, cfg_id, reduced: bool):
    """Roofline record of the step kernel that serves workload `w`."""
    N, n, dtype = w.N, w.ncols, w.dtype
    sm_max_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(device).multi_processor_count
    kernel_path = pkg.chase_filter_kernel_path(N, n, dtype)
    is_f64 = dtype in (torch.complex128, torch.float64)
    frac_3x = None
    if kernel_path == 2:
        # tcgen05: per algorithmic product one kind::tf32 MMA (hi*hi) + one kind::f16 BF16 MMA over a doubled K
        # for both cross terms = 2 MMA units (CHASE_TF32_MIXED=0: classic 3xTF32, 3 units).  The
        # peak for ALGORITHMIC flops is the TF32 tensor peak / units; TF32 peak = measured bf16 GEMM x nominal ratio.
        bf16, src = measured_bf16_sustained_tflops()
        units = 3.0 if os.environ.get("CHASE_TF32_MIXED", "1")[:1] == "0" else 2.0
        peak = bf16 * TF32_OVER_BF16_NOMINAL / units
        frac_3x = achieved_tflops / (bf16 * TF32_OVER_BF16_NOMINAL / 3.0)
        bound, kname = "tensor", "step_tf32_pair_kernel"
        peak_source = (f"{src} x nominal tf32/bf16 ratio {TF32_OVER_BF16_NOMINAL:.3f} / {units:.0f} MMA units per "
                       f"product ({'TF32 hi*hi + one BF16 MMA for both cross terms' if units == 2.0 else '3xTF32 split'}, "
                       f"DESIGN.md 6.4); power-capped part: sw_power_cap is expected")
    else:
        per_clk = FP64_FLOP_PER_CLK_SM * (1 if is_f64 else 2)     # FP32 FMA pipe: 256 flop/clk/SM
        peak = sms * per_clk * sm_max_mhz * 1e6 * 1e-12            # TFLOP/s
        bound = "tensor" if kernel_path == 1 else "alu"
        kname = "step_dmma_kernel" if kernel_path == 1 else "step_generic_kernel"
        peak_source = (f"{sms} SMs x {per_clk} flop/clk/SM x clocks.max.sm {sm_max_mhz:.0f} MHz "
                       f"(DESIGN.md 'Peak'); MEASURED_PEAKS.json has no FP64 entry")
    # DRAM bytes (read + write) of ONE full-width launch from the committed `ncu --set full` capture
    # (profiles/); only known for the two captured workloads.
    traffic, traffic_note = None, None
    if not reduced and cfg_id in NCU_TRAFFIC:
        traffic, traffic_note = NCU_TRAFFIC[cfg_id]
    return {
        "bound": bound, "kernel": kname,
        "achieved": achieved_tflops, "peak": peak, "unit": "TFLOP/s", "frac": achieved_tflops / peak,
        "traffic": traffic, "traffic_note": traffic_note, "peak_source": peak_source,
        "frac_of_nvidia_quoted_40tf": achieved_tflops / 40.0 if is_f64 else None,
        "frac_of_3xtf32_peak": frac_3x,
        # single-precision configs also against the FP32 FMA pipe (148 SMs x 256 flop/clk at max clock,
        # 74.5 TFLOP/s nominal) -- what a kernel WITHOUT tensor cores could reach at best
        "frac_of_fp32_fma_peak": (achieved_tflops / (sms * 2 * FP64_FLOP_PER_CLK_SM * sm_max_mhz * 1e-6)
                                  if not is_f64 else None),
        "algorithmic_flops_per_step": w.flops(), "launches_per_step": launches_per_step,
    }


def parity_vs_oracle(pkg, w, V_full, device, max_full_flops: float = 1.5e12):
    """GPU result of the FULL run (V_full, every column filtered with its own degree inside the timed
    launch configuration) against the oracle: the whole block when the oracle finishes in seconds,
    else the SURVEY 8(c) column sample (>= 32 columns, each with its own degree, full H; pin P7)."""
    import oracle
    N, n = w.N, w.ncols
    Hn = host_colmajor_numpy(w.H)
    if w.flops() <= max_full_flops:
        cols = list(range(n))
        sample = f"all {n} columns, full {N}x{N} H, own degrees"
    else:
        cols = W.parity_sample_columns(w.degrees)
        sample = (f"sampled: {len(cols)} of {n} columns (first/last of every degree class, tile edges, seeded random), "
                  f"full {N}x{N} H, own degrees")
    deg = w.degrees.numpy()[cols]
    Vs = host_colmajor_numpy(W.as_colmajor(w.V0[:, cols]))
    t0 = time.perf_counter()
    ref = oracle.chase_filter(Hn, Vs, deg, w.a, w.b, w.lambda1)
    dt = time.perf_counter() - t0
    del Hn
    got = host_colmajor_numpy(W.as_colmajor(V_full[:, cols]))
    col_err = np.linalg.norm(got - ref, axis=0) / np.linalg.norm(ref, axis=0)
    tol = 1e-12 if w.dtype in (torch.complex128, torch.float64) else 1e-4
    rel = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
    return {"rel_fro_vs_oracle": rel, "worst_column_rel_err": float(col_err.max()), "tolerance": tol,
            "ok": bool(rel <= tol), "sample": sample, "degrees_sampled": sorted(set(int(d) for d in deg)),
            "oracle_seconds": dt}


def cpu_blas_context(w, ncols: int = 128):
    """Context only: ONE step (H - cI) X through numpy's BLAS GEMM on the host cores, on a
    column block wide enough to be compute-bound -- what the paper's CPU path (ZHEMM, Listing 2) would
    achieve here.  Not the oracle, not the reference arm; labelled as such."""
    Hn = host_colmajor_numpy(w.H)
    X = np.asfortranarray(host_colmajor_numpy(W.as_colmajor(w.V0[:, :min(ncols, w.ncols)])))
    f = 8.0 if np.iscomplexobj(Hn) else 2.0
    t0 = time.perf_counter()
    Y = Hn @ X
    Y -= 0.5 * (w.a + w.b) * X
    dt = time.perf_counter() - t0
    return {"what": "numpy (vendor BLAS) GEMM, one step (H - cI) X, context only", "ncols": X.shape[1],
            "seconds": dt, "gflops": f * float(w.N) ** 2 * X.shape[1] / dt * 1e-9}


ALL_CONFIG_STEPS = {1: 1000, 2: 20, 3: 5, 5: 3}     # timed filter calls per non-headline config (3 warm-ups each)


def run_other_configs(pkg, device, headline_cfg: int):
    """The other BASELINE.json configs, each timed the same way as the headline one (own clock record)
    and compared with the oracle at full size: driver-observed numbers for cfgs 1, 2, 3, 5."""
    out = {}
    for cfg, steps in ALL_CONFIG_STEPS.items():
        if cfg == headline_cfg:
            continue
        try:
            w = W.make_config(cfg, device=device)
            r = time_filter(pkg, w, steps, 3, device, 1, 0, device.index or 0)
            value = w.flops() * steps / r["dev_s"] * 1e-9
            roof = roofline_of(pkg, w, value * 1e-3, r["clocks"], device, r["launches"] // steps, cfg, False)
            par = parity_vs_oracle(pkg, w, r["V"], device)
            out[f"cfg{cfg}"] = {
                "workload": f"N={w.N} {W.DTYPE_NAMES[w.dtype]}, V0 {w.N}x{w.ncols}, degrees "
                            f"{int(w.degrees.min())}..{int(w.degrees.max())}, sum_deg={w.sum_deg}",
                "value": value, "unit": UNIT, "steps": steps, "warmup": 3,
                "ms_per_step": r["dev_s"] / steps * 1e3, "ms_min": min(r["ms"]), "dtype": DTYPE_LABEL[w.dtype],
                "roofline": roof, "clocks": r["clocks"], "gpu_launches": r["launches"],
                "rel_fro_vs_oracle": par["rel_fro_vs_oracle"], "parity": par,
            }
            del r, w
        except Exception as exc:                       # one config failing must not lose the headline line
            out[f"cfg{cfg}"] = {"error": f"{type(exc).__name__}: {str(exc)[:300]}"}
        torch.cuda.empty_cache()
    return out


# Shapes whose column stride is not a multiple of 16 bytes cannot be described to TMA and run on the FMA kernels
# (kernel path 0): one large odd-N shape per precision, so that this path has a driver-observed throughput and a
# fraction of ITS roofline, the FP64 / FP32 FMA pipe: 148 SMs x 64 (128) FMA lanes x 2 flop x the max SM clock.
FMA_FALLBACK_SHAPES = {"f64_N20001": (3, 20001, 700), "c64_N30001": (5, 30001, 750)}
# dram bytes of one launch at exactly these shapes, from profiles/ncu_r3_step_generic.md (typed in, not measured here)
FMA_FALLBACK_TRAFFIC = {"f64_N20001": 30.101692e9 + 0.112300e9, "c64_N30001": 88.987575e9 + 0.190287e9}


def run_fma_fallback(pkg, device, sm_max_mhz: float):
    out = {}
    for name, (cfg, N, ncols) in FMA_FALLBACK_SHAPES.items():
        try:
            w = W.make_config(cfg, device=device, N=N, ncols=ncols)
            path = pkg.chase_filter_kernel_path(w.N, w.ncols, w.dtype)
            steps = 2
            r = time_filter(pkg, w, steps, 3, device, 1, 0, device.index or 0)
            tflops = w.flops() * steps / r["dev_s"] * 1e-12
            lanes = 64 if w.dtype in (torch.float64, torch.complex128) else 128
            peak = 148 * lanes * 2 * sm_max_mhz * 1e6 * 1e-12
            par = parity_vs_oracle(pkg, w, r["V"], device)
            out[name] = {
                "workload": f"N={w.N} {W.DTYPE_NAMES[w.dtype]}, V0 {w.N}x{w.ncols}, uniform degree {int(w.degrees.max())} "
                            f"(cfg {cfg}'s generator at an odd N)",
                "kernel_path": path, "value": tflops * 1e3, "unit": UNIT, "steps": steps, "warmup": 3,
                "ms_per_step": r["dev_s"] / steps * 1e3, "dtype": DTYPE_LABEL[w.dtype],
                "roofline": {"bound": "alu", "kernel": "step_generic_kernel", "achieved": tflops, "peak": peak,
                             "unit": "TFLOP/s", "frac": tflops / peak, "traffic": FMA_FALLBACK_TRAFFIC.get(name),
                             "traffic_note": "bytes of one launch; from profiles/ncu_r3_step_generic.md, not measured "
                                             "in this run",
                             "peak_source": f"148 SMs x {lanes} FMA lanes x 2 flop x {sm_max_mhz:.0f} MHz"},
                "clocks": r["clocks"], "gpu_launches": r["launches"],
                "rel_fro_vs_oracle": par["rel_fro_vs_oracle"], "parity": par,
            }
            del r, w
        except Exception as exc:
            out[name] = {"error": f"{type(exc).__name__}: {str(exc)[:300]}"}
        torch.cuda.empty_cache()
    return out


def run_ours(args):
    import paper_1805_10121_b200 as pkg
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    pkg.load()
    rank, world, local = dist_setup(args.gpus)
    device = torch.device("cuda", local)
    torch.cuda.set_device(device)

    w = build_workload(args, device, rank)
    N, n, dtype = w.N, w.ncols, w.dtype
    flops_step = w.flops()
    r = time_filter(pkg, w, args.steps, args.warmup, device, world, rank, local)
    V, launches, clocks, t_wall = r["V"], r["launches"], r["clocks"], r["t_wall"]
    r_ms = list(r["ms"])
    dev_s = max_over_ranks(r["dev_s"], world)
    total_flops = sum_over_ranks(flops_step * args.steps, world)
    value = total_flops / dev_s * 1e-9

    # ---- roofline of the step kernel (all launches of a step are the same kernel) --------------
    is_f64 = dtype in (torch.complex128, torch.float64)
    achieved = flops_step * args.steps / r["dev_s"] * 1e-12
    reduced = args.N is not None or args.ncols is not None
    roofline = roofline_of(pkg, w, achieved, clocks, device, launches // max(args.steps, 1), args.config, reduced)
    probe_dmma = pkg.chase_fp64_peak_probe(1, 1 << 16) * 1e-3
    probe_dfma = pkg.chase_fp64_peak_probe(0, 1 << 16) * 1e-3
    roofline.update({"peak_probe_dmma_tflops": probe_dmma, "peak_probe_dfma_tflops": probe_dfma,
                     "frac_of_probe_dmma": achieved / probe_dmma if is_f64 else None})

    # ---- parity of the timed configuration (rank 0, N = 1): the last timed run's V vs the oracle ----
    # ---- cpu_baseline: the oracle, as it stands, on a BOUNDED sample (about 10-30 s of CPU work) ----
    cpu_baseline, parity, blas_ctx = None, None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        parity = parity_vs_oracle(pkg, w, V, device)
        cols = sample_columns(w, args.sample_cols)
        Hn = host_colmajor_numpy(w.H)
        Vs = W.as_colmajor(w.V0[:, cols])
        dt, fl, _ = oracle_sample_run(Hn, host_colmajor_numpy(Vs), args.sample_degree, w)
        del Hn
        sample = (f"{len(cols)} of {n} columns (evenly spaced), full {N}x{N} H, degree truncated to "
                  f"{args.sample_degree}")
        cpu_baseline = {"value": fl / dt * 1e-9, "unit": UNIT, "cores": oracle.num_threads(), "nproc": os.cpu_count(), "kind": "oracle",
                        "sample": sample, "seconds": dt,
                        "extrapolated_seconds_for_the_whole_workload": dt * flops_step / fl}
        try:
            blas_ctx = cpu_blas_context(w)
        except Exception as exc:
            blas_ctx = {"error": str(exc)[:200]}

    # ---- aux: the other entry points on the same workload, device-timed --------------
    aux = None
    if rank == 0 and world == 1 and not args.no_aux:
        aux = time_aux_ops(pkg, w, V, device)

    # ---- comparator (context, not a dependency): one full-width H @ V0 through torch.matmul = cuBLAS ------
    comparator = None
    if rank == 0 and world == 1 and not args.no_aux:
        try:
            f = 8.0 if dtype.is_complex else 2.0
            out = torch.matmul(w.H, w.V0)          # warm-up (also picks the cuBLAS algorithm)
            torch.cuda.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record()
            out = torch.matmul(w.H, w.V0)
            c1.record()
            torch.cuda.synchronize()
            ms = c0.elapsed_time(c1)
            comparator = {"what": "torch.matmul(H, V0), all columns, no epilogue (cuBLAS GEMM on the same box)",
                          "ms": ms, "gflops": f * N * N * n / ms * 1e-6,
                          "ours_full_width_step_gflops": (aux or {}).get("chase_hemm", {}).get("gflops")}
            del out
        except RuntimeError as exc:                 # e.g. out of memory: context only
            comparator = {"error": str(exc)[:200]}

    # ---- e2e: HOST buffers through chase_filter_host (H2D + filter + D2H inside the timed call) --
    e2e = None
    if not args.no_e2e:
        Hh = torch.empty((N, N), dtype=dtype, pin_memory=True)
        Hh.copy_(w.H.t())
        Vh = torch.empty((n, N), dtype=dtype, pin_memory=True)
        Vh.copy_(w.V0.t())
        torch.cuda.synchronize()
        barrier(world)
        t0 = time.perf_counter()
        pkg.chase_filter_host(Hh.t(), Vh.t(), w.degrees, w.a, w.b, w.lambda1, device=local)
        barrier(world)
        e2e_s = max_over_ranks(time.perf_counter() - t0, world)
        h2d = Hh.numel() * Hh.element_size() + Vh.numel() * Vh.element_size()
        d2h = Vh.numel() * Vh.element_size()
        e2e = {"value": sum_over_ranks(flops_step, world) / e2e_s * 1e-9, "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": 1, "seconds": e2e_s,
               "api": "chase_filter_host (pinned host H, V; cudaMalloc + H2D + filter + D2H + free inside)"}
        del Hh, Vh

    # ---- the other BASELINE.json configs, driver-observed (rank 0, N = 1, default workload only) --------
    all_configs = None
    if rank == 0 and world == 1 and not args.no_all_configs and not reduced:
        cfg_line = workload_config(args, w, world)
        del V, r
        w.H = None
        w.V0 = None
        torch.cuda.empty_cache()
        all_configs = run_other_configs(pkg, device, args.config)
        all_configs["fma_fallback"] = run_fma_fallback(pkg, device, float((clocks or {}).get("sm_max_mhz") or 1965.0))
    else:
        cfg_line = workload_config(args, w, world)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_s / args.steps * 1e3, "ms_min": min(r_ms),
            "ms_median": statistics.median(r_ms), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": DTYPE_LABEL[dtype],
            "data": "synthetic", "config": cfg_line, "clocks": clocks,
            "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "parity": parity, "aux_ops": aux, "comparator_cublas": comparator, "cpu_blas_context": blas_ctx,
            "all_configs": all_configs, "wall_s_timed_region": t_wall,
            "fraction_of_fp64_peak": roofline["frac"] if is_f64 else None,
        }
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
