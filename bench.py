#!/usr/bin/env python
"""bench.py - the headline metric of BASELINE.json: fp64 likelihood evaluations / second.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl ours|reference]
                  [--dtype f64|f32] [--scaling weak|strong]

A "step" is one pass of the whole hot path (residual, forward FFT, generator product, inverse
FFT, fused quadratic reduction, summed over segments) over one batch of B synthetic templates
of the named config; the default workload is config c2 (N = 4096, B = 4096), the one the
metric is quoted on.  With --gpus N > 1 (launched by torchrun) every rank processes its own
batch of B templates (weak scaling, no data-path collective: templates are independent).

Prints ONE JSON line (rank 0).  Keys follow the driver's contract; see DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 likelihood evals/sec"
UNIT = "evals/s"
# fp64 ALU roofline: 64 DFMA/clk/SM x 148 SMs x 1.965 GHz x 2 flop (guide unit counts and
# clocks.max.sm); the register-loop DFMA / DMMA throughputs are measured in every run
# (libtdprobe.so, include/tdprobe.h) and reported beside it.  DESIGN.md 6.
FP64_PEAK_TFLOPS = 37.2
# fp32 evaluation mode (--dtype f32, never the headline): 128 FFMA/clk/SM x 148 SMs x 1.965 GHz x 2 flop
FP32_PEAK_TFLOPS = 74.4

def _dominant(seg_lengths, variant, f32):
    """Name of the FFT-path kernel that serves the longest segment (the dominant kernel of a step)."""
    n = int(max(seg_lengths))
    log2m = max(8, int(math.ceil(math.log2(max(n, 1)))))
    tail = " (fp32 build)" if f32 else ""
    if variant == 2:
        return "staged lg_* kernels" + tail
    if log2m <= 9:
        return f"td_fused_kernel<{log2m}>"
    if log2m <= 12:
        return f"td_fused4_kernel<{log2m}>" + tail
    if log2m == 13:
        return "td_cluster_kernel" + tail
    if log2m <= 16:
        if variant == 3 and log2m == 16 and not f32:
            return "td_cluster16_kernel"
        return f"td_group_kernel<{1 << (log2m - 12)}>" + tail
    return "staged lg_* kernels" + tail


def alg_flops_per_eval(seg_lengths) -> float:
    """three real length-m FFT equivalents + 2 half-spectrum products + O(N) tail."""
    tot = 0.0
    for n in seg_lengths:
        m = 2 * (1 << max(8, int(math.ceil(math.log2(max(int(n), 1))))))
        tot += 3 * 2.5 * m * math.log2(m) + 6 * m + 5 * int(n)
    return tot


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        rows = [r for (ts, r) in self.rows if t0 - 0.05 <= ts <= t1 + 0.1] or [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_rate(w, budget_templates: int):
    """The oracle as it stands on the host cores: (evals/s of the batched solve, factor seconds, cores, sample)."""
    from oracle import td_oracle as O
    try:
        from threadpoolctl import threadpool_info
        th = max([p.get("num_threads", 1) for p in threadpool_info()] or [os.cpu_count() or 1])
    except Exception:
        th = os.cpu_count() or 1
    nb = min(w.B, budget_templates)
    t0 = time.perf_counter()
    if w.n_tot > 40000 and len(w.seg_lengths) == 1:
        out = O.loglike_batch_solve_toeplitz(w.acf, w.seg_lengths, w.d, w.H[:nb])
        tf, ts = 0.0, time.perf_counter() - t0
        kind = "scipy solve_toeplitz per template (dense C does not fit)"
    else:
        fac = O.factorize(w.acf, w.seg_lengths)
        tf = time.perf_counter() - t0
        t1 = time.perf_counter()
        out = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H[:nb], factors=fac)
        ts = time.perf_counter() - t1
        kind = "Cholesky once (%.2f s, not counted) + batched forward substitution" % tf
    return nb / ts, tf, th, f"{nb} of {w.B} templates of {w.name}; {kind}", out


def gsce_rate(w, nb: int, ref: np.ndarray):
    """The paper's own fast CPU method (GSCE, Eqs. 14-16: Levinson once, then one forward and two inverse real FFTs per
    template with numpy's FFT; oracle/td_oracle.py, pin P20) on the same sample: the O(N log N) context line."""
    from oracle import td_oracle as O
    t0 = time.perf_counter()
    fac = O.gsce_factors(w.acf, w.seg_lengths)
    tf = time.perf_counter() - t0
    t1 = time.perf_counter()
    out = O.loglike_batch_gsce(w.acf, w.seg_lengths, w.d, w.H[:nb], factors=fac)
    ts = time.perf_counter() - t1
    err = float(np.max(np.abs(out - ref[:nb]) / np.maximum(np.abs(ref[:nb]), 1.0))) if ref is not None else None
    return {"value": nb / ts, "unit": UNIT, "kind": "oracle GSCE route: Levinson once (%.2f s, not counted) + numpy FFT circulant "
            "embedding per template (PAPER.md:231-254); single-threaded numpy FFT" % tf, "sample": f"{nb} templates",
            "max_rel_diff_vs_cholesky_route": err}


def run_reference(args):
    from paper_2603_06010_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nb = {"c1": 64, "c2": 1024, "c3": 256, "c4": 2, "c5": 256}.get(args.config, 256)
    w = W.make(args.config, B=nb)
    rates = []
    for i in range(args.warmup + args.steps):
        r, tf, th, sample, _ = oracle_rate(w, nb)
        if i >= args.warmup:
            rates.append(r)
    val = float(np.mean(rates))
    line = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * nb / val, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": f"{args.config}: bounded sample, each step = {sample}"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": th, "host_cpu_count": os.cpu_count(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="c2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--B", type=int, default=None, help="override templates per GPU (default: the config's B)")
    ap.add_argument("--n-scale", type=int, default=1,
                    help="divide every segment length of the config by this (workloads.make: the reduced-size versions the "
                         "parity tests use; profiling of the size classes between the configs, never the headline)")
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 FFT, 2 dense (Gohberg-Semencul), 4 CDO (cached L^-1)")
    ap.add_argument("--fft-variant", type=int, default=0)
    ap.add_argument("--op", default="loglike", choices=["loglike", "dh"],
                    help="loglike: the headline hot path; dh: only the cross term <d|h_b> (td_inner_batch, out_hh = NULL)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"],
                    help="f64: the headline; f32: fp32 evaluation with fp64 setup (td_set_precision, PAPER.md:322-324) - "
                         "a second line with its own fp32-FMA roofline, never the headline")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="--gpus N > 1: weak = every rank its own batch of B (default); strong = ONE batch of B sharded "
                         "over the ranks with shard.row_slice (no data-path collective either way)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--probe-peaks", action="store_true",
                    help="print the measured fp64 DFMA / DMMA / DADD register-loop throughputs and exit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2603_06010_b200 import binding as tdb
    from paper_2603_06010_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback exists)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    tdb.load(build_if_missing=False)
    if args.probe_peaks:
        if rank == 0:
            names = {0: "dfma", 1: "dmma_m8n8k4", 2: "dfma_and_dmma_interleaved", 3: "dadd", 4: "ffma_fp32"}
            print(json.dumps({"tflops": {names[k]: tdb.probe_throughput(k, local) for k in range(5)},
                              "derived_fp64_peak": FP64_PEAK_TFLOPS}))
        return

    w = W.make(args.config, B=args.B, n_scale=args.n_scale)
    B_job, n_tot = w.B, w.n_tot
    lo, hi = 0, B_job
    if world > 1 and args.scaling == "strong":
        from paper_2603_06010_b200 import shard
        lo, hi = shard.row_slice(B_job, rank, world)     # this rank's rows of the ONE batch
        w.H = w.H[lo:hi]
        if w.params is not None:
            w.params = w.params[lo:hi]
    B = hi - lo                                          # templates this rank evaluates per step
    units_per_step = B_job if (world > 1 and args.scaling == "strong") else world * B
    t_setup = time.perf_counter()
    h = tdb.TDLikelihood(w.acf, w.seg_lengths, device=local)   # S0: Levinson-Durbin + generator spectra, once per handle
    t_setup = time.perf_counter() - t_setup
    if args.path:
        h.set_path(args.path)
    if args.fft_variant:
        h.set_fft_variant(args.fft_variant)
    if args.dtype == "f32":
        try:
            h.set_precision(tdb.TD_PREC_F32)
        except tdb.TDError as e:
            if rank == 0:   # no size class of this config has an fp32 kernel (c4: staged kernels are fp64 only)
                print(json.dumps({"metric": "fp32-evaluation likelihood evals/sec", "dtype": "f32", "unavailable":
                                  f"{args.config}: td_set_precision(TD_PREC_F32) -> {e}"}))
            if world > 1:
                dist.destroy_process_group()
            return
    d = torch.as_tensor(w.d).to(dev)
    H_host = torch.as_tensor(w.H).pin_memory()
    # >= 3 distinct device copies of H, rotated, so no step is served from the 126 MB L2
    nbuf = max(3, int(math.ceil(3 * 126e6 / (8.0 * max(B, 1) * n_tot))))
    nbuf = min(nbuf, 64)
    Hs = [H_host.to(dev, non_blocking=True) for _ in range(nbuf)]
    out = torch.empty(B, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()

    if args.op == "dh":
        def step(Hd):
            h.inner_batch(d, Hd, want_hh=False, out_dh=out)
        args.no_e2e = True
    else:
        def step(Hd):
            h.loglike_batch(d, Hd, out=out)

    # ---------------- device-resident throughput
    # (the clock sampler starts BEFORE the warm-up steps: its start-up pause used to sit between warm-up and timed region,
    # and a GPU that has idled for 0.1 s runs its next few steps 1-30 % slower - the warm-up must be what directly precedes
    # the timed steps)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.12)
    barrier()
    for i in range(args.warmup):
        step(Hs[i % nbuf])
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches = 0
    torch.cuda.synchronize()
    barrier()
    t_wall0 = time.time()
    evs[0].record(stream)
    for i in range(args.steps):
        step(Hs[i % nbuf])
        launches += h.last_launches()
        evs[i + 1].record(stream)
    torch.cuda.synchronize()
    t_wall1 = time.time()
    barrier()
    total_ms = evs[0].elapsed_time(evs[-1])
    step_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)]
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    path_used = h.info()["last_path"]
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    value = units_per_step * args.steps / (total_ms * 1e-3)

    # ---------------- end to end: host buffers through the C ABI (H2D of H and d, D2H of out, per step)
    e2e = None
    if not args.no_e2e:
        # every host buffer of the end-to-end legs is page-locked (the contract: inputs come from pinned host memory)
        d_pin = torch.as_tensor(w.d).pin_memory().numpy()
        out_host = torch.empty(B, dtype=torch.float64).pin_memory().numpy()
        for _ in range(2):
            h.loglike_batch_host(d_pin, H_host, out_host)
        torch.cuda.synchronize()
        barrier()
        k_e2e = max(3, min(args.steps, 10))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(k_e2e):
            h.loglike_batch_host(d_pin, H_host, out_host)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        e2e = {"value": units_per_step * k_e2e / (ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(8 * B * n_tot + 8 * n_tot), "d2h_bytes_per_step": int(8 * B),
               "steps": k_e2e, "api": "td_loglike_batch_host (pinned H, chunked copies overlapped with kernels)"}
        max_dev = float(np.max(np.abs(out_host - out.cpu().numpy())))
        e2e["max_abs_diff_vs_device_call"] = max_dev

    # ---------------- the same evaluations from template PARAMETERS on the host (td_loglike_family_batch_host):
    # 5 doubles per template cross the bus, the rows are synthesised on the device.  Extra key, not `e2e`.
    e2e_params = None
    if not args.no_e2e and args.op == "loglike" and w.params is not None:
        d_pin = torch.as_tensor(w.d).pin_memory().numpy()
        p_pin = torch.as_tensor(np.ascontiguousarray(w.params)).pin_memory().numpy()
        out_p = torch.empty(B, dtype=torch.float64).pin_memory().numpy()
        for _ in range(2):
            h.loglike_family_batch_host(d_pin, w.family, p_pin, w.fs, out_p)
        torch.cuda.synchronize()
        barrier()
        k_p = max(3, min(args.steps, 10))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(k_p):
            h.loglike_family_batch_host(d_pin, w.family, p_pin, w.fs, out_p)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        e2e_params = {"value": units_per_step * k_p / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(8 * w.params.size + 8 * n_tot),
                      "d2h_bytes_per_step": int(8 * B), "steps": k_p,
                      "api": f"td_loglike_family_batch_host (host parameters, family {W.FAMILIES[w.family]}; templates synthesised on the device)",
                      "max_rel_diff_vs_device_call": float(np.max(np.abs(out_p - out.cpu().numpy()) / np.maximum(np.abs(out_p), 1.0)))}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---------------- rooflines (dominant kernel = the one kernel of the step on the fused path)
    peaks, peaks_kind = measured_peaks()
    kern_ms = float(np.mean(step_ms))
    dense = path_used in (2, 4)
    cdo = path_used == 4   # triangular W = L^-1 contraction: N^2 flop per template and segment (half of the GS dense path)
    falg = (float(sum((1.0 if cdo else 2.0) * int(n) * int(n) for n in w.seg_lengths)) if dense
            else alg_flops_per_eval(w.seg_lengths))
    f32 = args.dtype == "f32"
    probe = {"dfma": tdb.probe_throughput(0, local), "dmma": tdb.probe_throughput(1, local)}
    if f32:
        probe["ffma_fp32"] = tdb.probe_throughput(4, local)
    peak_tf = FP32_PEAK_TFLOPS if f32 else FP64_PEAK_TFLOPS
    ach_tf = falg * B / (kern_ms * 1e-3) / 1e12
    ach_gbs = (8.0 * n_tot * B + 8.0 * B) / (kern_ms * 1e-3) / 1e9
    traffic, traffic_source = None, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp) and not f32:
        try:
            tj = json.load(open(tp))
            traffic = tj.get(args.config)
            traffic_source = ("a constant from a committed ncu capture, NOT a counter of this run: " +
                              tj.get("_source", "profiles/traffic.json")) if traffic is not None else None
        except Exception:
            traffic = None
    roofline = {"bound": "tensor" if dense else "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf,
                # fraction against the DFMA register loop measured in THIS run (state both denominators)
                "frac_vs_measured_loop": ach_tf / probe["ffma_fp32" if f32 else "dfma"],
                "traffic": traffic, "traffic_source": traffic_source,
                "kernel": ("td_cdo_kernel" if cdo else "td_dense_kernel") if dense else _dominant(w.seg_lengths, args.fft_variant, f32),
                "measured_register_loop_tflops": probe,
                "kernel_ms": kern_ms, "alg_flops_per_eval": falg,
                "peak_source": ("derived: 128 FFMA/clk/SM x 148 SM x 1.965 GHz x 2; the FFMA register loop of this run beside it"
                                if f32 else
                                "derived: 64 DFMA/clk/SM x 148 SM x 1.965 GHz x 2 (DESIGN.md 6); the fp64 tensor pipe "
                                "(DMMA.8x8x4) has the same peak; register-loop measurements of this run beside it")}
    if args.op == "dh":
        # the cross term is one streaming pass over H: HBM is the bounding roofline; 2 flop per 8 bytes
        roofline = {"bound": "hbm", "achieved": ach_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": ach_gbs / peaks["hbm_gbs"], "traffic": None, "kernel": "dot_rows_kernel",
                    "kernel_ms": kern_ms, "peak_source": peaks_kind + " (MEASURED_PEAKS.json copy bandwidth); the step also "
                    "holds the once-per-call setup kernels (z of d, weights u = C^-1 d)"}
        args.no_cpu_baseline = True
    roofline_hbm = {"bound": "hbm", "achieved": ach_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": ach_gbs / peaks["hbm_gbs"], "peak_source": peaks_kind + " (MEASURED_PEAKS.json copy bandwidth)",
                    "alg_bytes_per_eval": 8.0 * n_tot + 8.0}

    # ---------------- the oracle on the host cores, bounded sample
    cpu = None
    if not args.no_cpu_baseline:
        budget = {"c1": 64, "c2": 2048, "c3": 256, "c4": 2, "c5": 256}.get(args.config, 256)
        r, tf, th, sample, ref = oracle_rate(w, budget)
        got = out.cpu().numpy()[: len(ref)]
        cpu = {"value": r, "unit": UNIT, "cores": th, "host_cpu_count": os.cpu_count(), "kind": "oracle",
               "note": "the oracle is the O(N^2)-per-template dense Cholesky route (fp64), not the paper's O(N log N) GSCE "
                       "route: a ratio against it is a ratio against a deliberately plain program",
               "sample": sample,
               "max_rel_err_gpu_vs_oracle": float(np.max(np.abs(got - ref) / np.maximum(np.abs(ref), 1.0))),
               "gsce": gsce_rate(w, len(ref), ref)}

    metric = METRIC if args.op == "loglike" else "fp64 cross-term <d|h_b> evals/sec (not the headline)"
    if f32:
        metric = "fp32-evaluation likelihood evals/sec (fp64 setup; second line, not the headline)"
    line = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": f"{args.config}: {w.description}; N_tot={n_tot}, segments={list(map(int, w.seg_lengths))}, "
                                   + (f"B={B_job} sharded over {world} GPUs (rank 0: {B})" if args.scaling == "strong" and world > 1
                                      else f"B={B} per GPU"),
                       "path": {1: "fft", 2: "dense", 3: "dot", 4: "cdo"}.get(path_used, "?"),
                       "l2": f"{nbuf} distinct device copies of H rotated between steps (H = {8 * B * n_tot / 2**20:.0f} MiB each)",
                       "parallelism": f"dp{world} over templates",
                       "setup_ms_not_in_metric": round(1e3 * t_setup, 3)},
            "roofline": roofline, "roofline_hbm": roofline_hbm, "cpu_baseline": cpu, "e2e": e2e, "e2e_params": e2e_params,
            "gpu_launches": launches, "clocks": clocks}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
