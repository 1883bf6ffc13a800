"""bench.py -- throughput of the HELIOS two-stream hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch: one radiative-equilibrium iteration
(a0-a9: level temperatures, k-table interpolation, Planck, sublayer optics, 1+n_scat sweeps,
quadrature/bolometric reduction, temperature update) of every column of the workload, i.e. one
helios_iterate_re(ctx, 1, ...) call.  Default workload: BASELINE.json configs[4] (8192 columns x
1000 bins x 20 g x 100 layers, scattering on, n_scat = 4), the configuration the metric's target
is quoted on.  N > 1: every rank runs its own 8192-column shard (weak scaling, no data-path
collective: columns are independent).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--cols M]

--impl reference times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample of the
same workload.  One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1606_05474_b200 import inputs  # noqa: E402

METRIC = "(bin*g*layer) two-stream flux updates/s"
UNIT = "updates/s"
# Algorithmic FP64 work per (bin, g, layer) update with n_scat = 4 (SURVEY.md
# section 8(d)): ~220 issued DP instructions, counted as FMA-equivalents (2 flop each).
DP_INSTR_PER_UPDATE_NSCAT4 = 220.0
# From the ncu --set full captures of the build being benchmarked (profiles/r2_k_flux_fp64_ncu.md,
# profiles/r2_k_flux_fp32_ncu.md; one k_flux launch at the default workload).  They are stored, not re-measured by
# this run (a number taken under a profiler is never a bench value); the line says where they come from.
#   traffic:  dram__bytes_read.sum + dram__bytes_write.sum
#   executed: lane instructions per update actually issued on the arithmetic pipes (DFMA+DMUL+DADD, resp.
#             FFMA+FMUL+FADD + 2 x (FFMA2+FMUL2+FADD2), packed instructions counted as two), from the SASS opcode
#             histogram of the same capture
NCU_PROFILE = {
    ("fp64", 4, 8192): {"traffic": 2.6344e8, "executed_instr_per_update": 167.2, "pipe_active_pct": 43.5,
                        "source": "profiles/r2_k_flux_fp64_ncu.md"},
    ("fp32", 4, 8192): {"traffic": 1.7006e8, "executed_instr_per_update": 167.1, "pipe_active_pct": 44.9,
                        "source": "profiles/r2_k_flux_fp32_ncu.md"},
}
FP64_LANES_PER_SM = 64
SM_COUNT = 148


def dp_instr_per_update(n_scat: int, any_scat: bool) -> float:
    """Survey table 8(d): 180 sweep-independent + 8 per sweep (4 FMA x 2 sublayers) per layer."""
    sweeps = 1 + (n_scat if any_scat else 0)
    return 180.0 + 8.0 * sweeps


def sp_instr_per_update(n_scat: int, any_scat: bool) -> float:
    """fp32 ray arithmetic: exp and reciprocals are single MUFU instructions, so
    the sweep-independent part is ~90 FP32 instructions per layer (kappa 8, dtau 6, 2 x [expm1 series 8,
    coefficients and sources 24], reduction 6, Planck share 18 in fp64 counted as issued) + 8 per sweep."""
    sweeps = 1 + (n_scat if any_scat else 0)
    return 90.0 + 8.0 * sweeps


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True,
                                     timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(cfg: int, cols, world: int, rank: int):
    base = inputs.make_config(cfg, n_cols=cols)
    nc = base.params["n_cols"]
    if world == 1:
        return base, nc
    full = inputs.make_config(cfg, n_cols=nc * world)          # every rank draws the same batch ...
    return full.take_columns(list(inputs.shard_columns(nc * world, rank, world))), nc   # ... and takes its shard


def oracle_sample(cfg: int, sample_cols: int, iters: int):
    """The oracle as it stands on a bounded sample: the first `sample_cols` columns x `iters` RE steps."""
    from oracle import binding as orc
    inp = inputs.make_config(cfg, n_cols=sample_cols)
    p = inp.params
    t0 = time.perf_counter()
    orc.iterate_re(inp, iters)
    dt = time.perf_counter() - t0
    updates = float(sample_cols) * p["n_bins"] * p["n_g"] * p["n_layers"] * iters
    return updates / dt, dt, orc.num_threads(), inp


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import binding as orc
    orc.build()
    cols = 16 if args.config == 4 else (8 if args.config == 3 else 1)
    it = 1
    oracle_sample(args.config, 1, 1)                        # page in
    times = []
    for _ in range(args.warmup):
        oracle_sample(args.config, cols, it)
    val = 0.0
    t_all = time.perf_counter()
    for _ in range(args.steps):
        v, dt, cores, inp = oracle_sample(args.config, cols, it)
        times.append(dt)
    total = time.perf_counter() - t_all
    p = inp.params
    upd = float(cols) * p["n_bins"] * p["n_g"] * p["n_layers"] * it * args.steps
    val = upd / sum(times)
    sample = f"first {cols} columns of config {args.config} x {it} RE iteration per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config}] (bounded sample: {sample})",
                       "n_layers": p["n_layers"], "n_bins": p["n_bins"], "n_g": p["n_g"], "n_scat": p["n_scat"]},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "wall_s": total}
    print(json.dumps(line), flush=True)


def measure_other_precision(args, inp, nc, updates_per_step, prec, any_scat, sm_max, direct=False):
    """Config 4 asks for fp64 and fp32: the same steps once more in the other arithmetic (N = 1).
    direct: the same steps with the direct coupled solve (n_scat = HELIOS_NSCAT_DIRECT, S12)
    instead of the 1 + n_scat sweeps; reported next to the headline, not as the headline."""
    import dataclasses
    import torch
    from paper_1606_05474_b200 import binding
    i2 = dataclasses.replace(inp, params=dict(inp.params, precision=1 if prec == "fp32" else 0))
    if direct:
        i2 = dataclasses.replace(i2, params=dict(i2.params, n_scat=binding.NSCAT_DIRECT))
    h = binding.Helios(i2, device="cuda:0")
    for _ in range(args.warmup):
        h.helios_iterate_re(1)
    h.helios_enable_timing(True)
    h.helios_kernel_time_ms()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(h.stream)
    for _ in range(args.steps):
        h.helios_iterate_re(1)
    e1.record(h.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    k_ms, k_n = h.helios_kernel_time_ms()
    h.close()
    p = inp.params
    f32 = prec == "fp32"
    if direct:
        return {"dtype": "f32" if f32 else "f64", "n_scat": "direct (HELIOS_NSCAT_DIRECT)",
                "value": updates_per_step * args.steps / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / args.steps,
                "kernel_ms": k_ms / max(k_n, 1),
                "note": "same workload, sweeps replaced by the direct solve of the coupled system (their n_scat -> infinity limit)"}
    instr = sp_instr_per_update(p["n_scat"], any_scat) if f32 else dp_instr_per_update(p["n_scat"], any_scat)
    lanes = 2 * FP64_LANES_PER_SM if f32 else FP64_LANES_PER_SM
    peak = 2.0 * SM_COUNT * lanes * sm_max * 1e6 / 1e12
    ach = 2.0 * instr * updates_per_step / (k_ms / max(k_n, 1) * 1e-3) / 1e12
    return {"dtype": "f32" if f32 else "f64", "value": updates_per_step * args.steps / (ms * 1e-3), "unit": UNIT,
            "ms_per_step": ms / args.steps,
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "alu_instr_per_update": instr, "kernel_ms": k_ms / max(k_n, 1)}}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1606_05474_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    inp, nc = workload(args.config, args.cols, world, rank)
    fp32 = args.precision == "fp32"
    if fp32:
        inp.params = dict(inp.params, precision=1)
    p = inp.params
    h = binding.Helios(inp, device=f"cuda:{local}")
    shape = h.helios_launch_shape()
    any_scat = bool(np.any(inp.w0 > 0))
    updates_per_step = float(nc) * p["n_bins"] * p["n_g"] * p["n_layers"]       # per rank

    def step():
        h.helios_iterate_re(1)

    for _ in range(args.warmup):
        step()
    barrier()
    l0 = h.helios_launch_count()
    h.helios_enable_timing(True)
    h.helios_kernel_time_ms()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(h.stream)
    for _ in range(args.steps):
        step()
    e1.record(h.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary() if rank == 0 else None
    k_ms, k_n = h.helios_kernel_time_ms()
    h.helios_enable_timing(False)
    launches = h.helios_launch_count() - l0
    if world > 1:
        t = torch.tensor([ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = updates_per_step * world * args.steps / (ms * 1e-3)

    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    T_host = torch.empty((nc, p["n_layers"]), dtype=torch.float64).pin_memory()
    it_host = torch.empty(nc, dtype=torch.int32).pin_memory()
    cv_host = torch.empty(nc, dtype=torch.int32).pin_memory()
    T_host.copy_(torch.from_numpy(np.ascontiguousarray(inp.T0)))
    T_np, it_np, cv_np = T_host.numpy(), it_host.numpy(), cv_host.numpy()
    h.helios_iterate_re_host(1, T_np, it_np, cv_np)            # warm
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        h.helios_iterate_re_host(1, T_np, it_np, cv_np)        # synchronous: H2D T, step, D2H T/iters/converged
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    if world > 1:
        t = torch.tensor([e2e_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    e2e_value = updates_per_step * world * args.steps / (e2e_ms * 1e-3)
    h2d = nc * p["n_layers"] * 8
    d2h = nc * p["n_layers"] * 8 + 2 * nc * 4

    if rank != 0:
        h.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (ray) kernel: FP64 ALU bound
    instr = sp_instr_per_update(p["n_scat"], any_scat) if fp32 else dp_instr_per_update(p["n_scat"], any_scat)
    lanes = 2 * FP64_LANES_PER_SM if fp32 else FP64_LANES_PER_SM
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tflops = 2.0 * SM_COUNT * lanes * sm_max * 1e6 / 1e12
    k_avg_ms = k_ms / max(k_n, 1)
    achieved = 2.0 * instr * updates_per_step / (k_avg_ms * 1e-3) / 1e12
    fma_meas = binding.helios_measure_fma_peak(binding.PREC_FP32 if fp32 else binding.PREC_FP64, h.stream.cuda_stream)
    fma3_meas = binding.helios_measure_fma3_peak(binding.PREC_FP32 if fp32 else binding.PREC_FP64, h.stream.cuda_stream)
    hbm_bytes = (inp.ktab.nbytes + nc * p["n_layers"] * 8 + nc * p["n_bins"] * 8 + 2 * nc * (p["n_layers"] + 1) * 8)
    prof = NCU_PROFILE.get((args.precision, args.config, nc), {})
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops,
                "traffic": prof.get("traffic"), "traffic_source": prof.get("source"),
                # frac counts the ALGORITHMIC instructions (220 per update at n_scat = 4); the kernel
                # issues fewer, so the share of the pipe's issue slots it really uses is lower:
                "executed_instr_per_update": prof.get("executed_instr_per_update"),
                "executed_frac": (achieved / peak_tflops * prof["executed_instr_per_update"] / instr) if prof else None,
                "executed_source": prof.get("source"),
                "kernel": "hx::k_flux", "kernel_ms": k_avg_ms, "kernel_launches": int(k_n),
                "kernel_share_of_step": k_ms / ms if ms > 0 else None,
                "alu_instr_per_update": instr,
                "peak_how": f"derived: {SM_COUNT} SMs x {lanes} {'FP32' if fp32 else 'FP64'} lanes x 2 flop x {sm_max:.0f} MHz (clocks.max.sm)",
                "fma_microbench_tflops": 2.0 * fma_meas / 1e12,
                "fma3_microbench_tflops": 2.0 * fma3_meas / 1e12,
                "frac_of_fma3_microbench": achieved / (2.0 * fma3_meas / 1e12) if fma3_meas > 0 else None,
                "frac_of_fma_microbench": achieved / (2.0 * fma_meas / 1e12) if fma_meas > 0 else None,
                "hbm_algorithmic_bytes": hbm_bytes,
                "hbm_time_floor_ms": 1e3 * hbm_bytes / (float(peaks.get("hbm_gbs", 6650.0)) * 1e9)}

    other = None
    if world == 1 and not args.no_other_precision:
        other = measure_other_precision(args, inp, nc, updates_per_step, "fp64" if fp32 else "fp32", any_scat, sm_max)

    direct = None
    if world == 1 and not args.no_other_precision and any_scat:
        direct = measure_other_precision(args, inp, nc, updates_per_step, args.precision, any_scat, sm_max, direct=True)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import binding as orc
        orc.build()
        s_cols, s_it = (64, 8) if args.config == 4 else ((64, 24) if args.config == 3 else (1, 400))   # ~15 s of oracle time
        v, dt, cores, _ = oracle_sample(args.config, s_cols, s_it)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {s_cols} columns of config {args.config} x {s_it} RE iterations ({dt:.1f} s)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if fp32 else "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config}]: {nc} columns/GPU x {p['n_bins']} bins x "
                                   f"{p['n_g']} g x {p['n_layers']} layers, n_scat={p['n_scat']}, one RE iteration per step",
                       "n_cols_per_gpu": nc, "n_layers": p["n_layers"], "n_bins": p["n_bins"], "n_g": p["n_g"],
                       "n_scat": p["n_scat"], "parallelism": f"columns sharded over {world} GPU(s), no collective",
                       "l2": f"inputs exceed L2 (k-table {inp.ktab.nbytes / 2**20:.0f} MiB + per-column arrays)",
                       "launch": shape},
            "re_iterations_per_s": {"batch": args.steps / (ms * 1e-3), "column": nc * world * args.steps / (ms * 1e-3)},
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": e2e_ms / args.steps, "api": "helios_iterate_re_host (pinned host buffers)"},
            "roofline": roofline, "cpu_baseline": cpu, "other_precision": other, "direct_solve": direct}
    print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--cols", type=int, default=None, help="override the number of columns per GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-precision", action="store_true",
                    help="skip the short measurement of the other arithmetic (fp32 next to fp64)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"],
                    help="arithmetic of the ray kernel (config 4 asks for both; fp64 is the default line)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
