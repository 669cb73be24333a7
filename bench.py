#!/usr/bin/env python
"""bench.py -- detector-samples/s of the gateau hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--variant default|fp32|tensor]
    python bench.py --impl reference ...      # the CPU oracle, timed on the host cores

One "step" = one pass of the whole hot path (geometry -> fused generator/contraction/photon
noise -> pink noise) over the full workload (default: BASELINE.json configs[3], the 61-spaxel
IFU config the metric and the roofline target are quoted on; it fits one GPU).  `value` is
timed with inputs and outputs resident in HBM; `e2e` runs the public API from HOST buffers
(pinned H2D of the inputs, gt_plan_create, gt_simulate streaming the TOD into pinned host
memory) inside the timed region.  With N > 1 (torchrun) every rank simulates an independent
observation (seed + rank) of the same config: weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "detector-samples/s"
UNIT = "detector-samples/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--variant", default="default", choices=["default", "fp32", "tensor"])
    ap.add_argument("--samples", type=int, default=None, help="shrink n_samples (debug only; marks the line invalid)")
    ap.add_argument("--shard", default="replica", choices=["replica", "spaxel"],
                    help="N > 1: 'replica' = independent observations per rank (weak scaling, the default); 'spaxel' = the "
                         "workload's spaxels split over the ranks, Kelvin output and the common-mode subtraction of Eq. 25 "
                         "with its one all-reduce over [t x chan] inside the step (strong scaling)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--peak-seconds", type=float, default=4.0, help="length of the sustained matmul runs that measure the tensor peaks")
    ap.add_argument("--no-peaks", action="store_true", help="skip the in-run measurement of the TF32 / fp16 / FP32 / PCIe denominators")
    ap.add_argument("--no-extras", action="store_true", help="skip the timing lines of the paper's own options (rows f1-f3)")
    ap.add_argument("--timeline", default=None, help="write the per-chunk compute / D2H timeline of one end-to-end step to this file")
    return ap.parse_args()


def workload_config(w, extra=None):
    cfg = {"workload": f"{w.name}: {w.n_spaxel} spaxel x {w.n_chan} chan x {w.n_samples} samples, "
                       f"{w.n_freq} freq, {len(w.stages)}-stage cascade, photon={int(w.photon_noise)} pink={int(w.pink_noise)}",
           "n_spaxel": w.n_spaxel, "n_chan": w.n_chan, "n_freq": w.n_freq, "n_samples": w.n_samples,
           "cache": "inputs (cube+screen) and the TOD written per step are larger than L2"}
    if extra:
        cfg.update(extra)
    return cfg


# ------------------------------------------------------------------------------------------
# clocks during the timed region (recipe's nvidia-smi line)
# ------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
                for nm, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference): the only places that execute oracle/
# ------------------------------------------------------------------------------------------
def oracle_sample(w, seconds):
    """Times the oracle, as it stands, on a bounded prefix of the workload (all spaxels and
    channels, the first n samples), sized for about `seconds` of wall time."""
    from oracle import oracle as O
    o = O.Oracle(w)
    cores = O.num_threads()
    per_sample = w.n_spaxel * w.n_chan
    n = max(1, min(w.n_samples, 4096 // max(w.n_spaxel, 1)))
    t0 = time.perf_counter(); o.simulate(0, n, want=("tod",)); dt = time.perf_counter() - t0
    if dt < 0.5 * seconds:
        n2 = int(min(w.n_samples, max(n, n * (seconds - dt) / max(dt, 1e-3))))
        t0 = time.perf_counter(); o.simulate(0, n2, want=("tod",)); dt = time.perf_counter() - t0
        n = n2
    return {"value": n * per_sample / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} samples x {w.n_spaxel} spaxels x {w.n_chan} channels of {w.name} "
                      f"({n * w.n_spaxel} rows, {dt:.1f} s wall, OpenMP over rows, fp64)"}, n, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2604_23305_b200 import workloads as W
    w = W.make_workload(args.workload, n_samples=args.samples)
    from oracle import oracle as O
    o = O.Oracle(w)
    cores = O.num_threads()
    # size one step at ~ (120 s / (steps + warmup)) of oracle work, from a short calibration
    n = max(1, 2048 // w.n_spaxel)
    t0 = time.perf_counter(); o.simulate(0, n, want=("tod",)); dt = time.perf_counter() - t0
    budget = 120.0 / max(args.steps + args.warmup, 1)
    n_step = int(max(1, min(w.n_samples, n * budget / max(dt, 1e-3))))
    for _ in range(args.warmup):
        o.simulate(0, n_step, want=("tod",))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.simulate(0, n_step, want=("tod",))
    total = time.perf_counter() - t0
    units = n_step * w.n_spaxel * w.n_chan * args.steps
    value = units / total
    sample = (f"each step = first {n_step} samples x {w.n_spaxel} spaxels x {w.n_chan} channels of {w.name} "
              f"({n_step * w.n_spaxel} rows), CPU oracle fp64, OpenMP")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, {"sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------
def peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return d, "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, \
        "fallback (B200_PROFILING.md)"


def measure_peaks(torch, B, dev, seconds):
    """The denominators SURVEY 8d asks to MEASURE, in this run and on this GPU: dense fp16 and TF32 matmul 8192^3
    (torch / cuBLAS is fine for a measurement: burst = best of 10, sustained = back to back for `seconds`), the FP32 FMA
    peak (the library's register-only loop), and the host link (1 GiB pinned cudaMemcpyAsync, both directions)."""
    out = {}
    n = 8192
    old = torch.backends.cuda.matmul.allow_tf32
    for name, dt, tf32 in (("f16", torch.float16, False), ("tf32", torch.float32, True)):
        torch.backends.cuda.matmul.allow_tf32 = tf32
        a = torch.randn((n, n), device=dev, dtype=dt); b = torch.randn((n, n), device=dev, dtype=dt)
        c = torch.empty((n, n), device=dev, dtype=dt)
        for _ in range(3):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); torch.matmul(a, b, out=c); e1.record(); e1.synchronize()
            best = max(best, 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k, t0 = 0, time.perf_counter()
        e0.record()
        while time.perf_counter() - t0 < seconds:
            for _ in range(20):
                torch.matmul(a, b, out=c)
            k += 20
            torch.cuda.synchronize()
        e1.record(); e1.synchronize()
        out[f"peak_{name}_measured"] = best
        out[f"peak_{name}_sustained_measured"] = 2.0 * n ** 3 * k / (e0.elapsed_time(e1) * 1e-3) / 1e12
        del a, b, c
    torch.backends.cuda.matmul.allow_tf32 = old
    out["peak_fp32_fma_measured"] = B.measure_fp32_fma()
    nb = 1 << 30
    host = torch.empty(nb, dtype=torch.uint8, pin_memory=True); devb = torch.empty(nb, dtype=torch.uint8, device=dev)
    for name, src, dst in (("d2h", devb, host), ("h2d", host, devb)):
        rates = []
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); dst.copy_(src, non_blocking=True); e1.record(); e1.synchronize()
            rates.append(nb / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        out[f"pcie_{name}_gbs"] = float(np.median(rates[1:]))
    del host, devb
    out["how"] = (f"torch.matmul {n}^3 fp16 and TF32 (allow_tf32): best of 10 and back to back for {seconds:g} s; FP32: "
                  "gt_measure_fp32_fma (register-only FMA loop); PCIe: median of 9 pinned 1 GiB copies per direction")
    return out


def ncu_traffic(kernel, rows_per_launch):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/*_traffic.csv),
    scaled by rows when bench's launch size differs from the captured one; None if there is no capture."""
    import csv
    best = None
    for f in sorted((ROOT / "profiles").glob("*_traffic.csv")):
        for r in csv.DictReader(open(f)):
            if r["kernel"] == kernel:
                best = r
    if best is None:
        return None, None
    per_row = (float(best["dram_bytes_read"]) + float(best["dram_bytes_write"])) / float(best["launch_rows"])
    return per_row * rows_per_launch, best["source"]


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2604_23305_b200 import binding as B
    from paper_2604_23305_b200 import workloads as W
    from paper_2604_23305_b200 import shard

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the gateau_b200 path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = W.make_workload(args.workload, n_samples=args.samples)
    variant = {"default": B.VARIANT_DEFAULT, "fp32": B.VARIANT_FP32, "tensor": B.VARIANT_TENSOR}[args.variant]
    if args.shard == "spaxel":
        return run_spaxel_sharded(args, torch, dist, B, W, shard, w, variant, rank, world, local, barrier)
    w = w.replace(seed=shard.replica_seed(w.seed, rank))          # independent observation per rank
    plan = B.Plan(w, variant=variant, device=f"cuda:{local}")
    units = w.detector_samples()
    tod = torch.empty((w.n_samples, w.n_spaxel, w.n_chan), dtype=torch.float32, device=f"cuda:{local}")

    for _ in range(max(args.warmup, 3)):
        plan.simulate(out=tod)
    barrier()
    sampler = ClockSampler(local); sampler.start()
    launches0 = plan.launch_count
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    fused_ms, fused_n = 0.0, 0
    barrier()
    step_ms = []
    for k in range(args.steps):
        ev[k].record()
        plan.simulate(out=tod)
        e = torch.cuda.Event(enable_timing=True); e.record(); e.synchronize()
        step_ms.append(ev[k].elapsed_time(e))
        ms, n = plan.last_fused_ms(); fused_ms += ms; fused_n += n
    barrier()
    total_ms = float(sum(step_ms))
    launches = plan.launch_count - launches0
    clocks = sampler.stop()
    total_ms = shard.max_over_ranks(total_ms, dist if world > 1 else None, device=f"cuda:{local}")
    value = shard.aggregate_throughput(units, world, args.steps, total_ms)

    # ---- roofline of the dominant kernel (the fused kernel) ----
    pk, pk_src = peaks()
    flops_per_launch = 2.0 * w.n_chan * w.n_freq * (w.n_samples * w.n_spaxel) / max(fused_n / args.steps, 1)
    avg_launch_s = fused_ms * 1e-3 / max(fused_n, 1)
    achieved = flops_per_launch / avg_launch_s / 1e12
    measured = {}
    if not args.no_peaks and rank == 0 and world == 1:
        try:
            measured = measure_peaks(torch, B, f"cuda:{local}", args.peak_seconds)
        except Exception as ex:                                   # report, never fake
            measured = {"error": repr(ex)[:200]}
    if plan.variant_name.startswith("tcgen05"):
        corr_blocks, corr_skipped = plan.corrections()
        issued_per_useful = 1.0 + 2.0 * (1.0 - corr_skipped / max(corr_blocks, 1))
        peak = pk["bf16_tflops_sustained"]                # the MMAs run as kind::f16 (fp16 rate = bf16 rate); kernel timed inside a long step: sustained figure
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": None, "kernel": "fused_tc_kernel",
                "peak_source": f"dense fp16/bf16 sustained (the dtype the MMAs run in), {pk_src}", "peak_burst": pk["bf16_tflops"],
                "mma_dtype": "f16 (three-term split of fp32 operands, fp32 accumulate)",
                "issued_tflops": issued_per_useful * achieved, "issued_frac": issued_per_useful * achieved / peak,
                "issued_per_useful": issued_per_useful, "corrections": {"products": int(corr_blocks), "skipped": int(corr_skipped)},
                "tf32_class_peak": measured.get("peak_tf32_sustained_measured") or 0.5 * peak,
                "tf32_class_peak_source": "measured in this run (torch TF32 matmul, sustained)" if measured.get("peak_tf32_sustained_measured")
                                          else "0.5 x fp16/bf16 sustained (nominal ratio)",
                "note": "achieved = algorithmic (useful) 2*n_chan*n_freq flop/row; frac = useful / fp16 peak.  issued_* counts the "
                        "fp16 products the split really issues per useful one: hi*hi always, lo*hi and hi*lo (kind::f16 K=16 MMAs) "
                        "only in the (column group, slab) blocks where the plan could not prove them negligible (banded "
                        "corrections: gt_debug_corrections): issued_per_useful = 1 + 2 (1 - skipped / products), at most 3.  "
                        "tf32_class_frac = useful flop against the TF32 dense peak, the denominator north_star names"}
        roof["tf32_class_frac"] = achieved / roof["tf32_class_peak"]
    else:
        mhz = clocks.get("sm_mhz") or pk.get("sm_max_mhz", 1965.0)
        peak = measured.get("peak_fp32_fma_measured") or 148 * 128 * 2 * mhz * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": None, "kernel": "fused_fp32_kernel",
                "peak_source": "FP32 FMA measured in this run (gt_measure_fp32_fma)" if measured.get("peak_fp32_fma_measured")
                               else f"FP32 FMA = 148 SM x 128 lanes x 2 x {mhz:.0f} MHz (median SM clock under load)"}
    roof.update({k: v for k, v in measured.items() if k.startswith("peak_")})
    if measured.get("how"):
        roof["measured_how"] = measured["how"]
    roof["traffic"], roof["traffic_source"] = ncu_traffic(roof["kernel"], (w.n_samples * w.n_spaxel) / max(fused_n / args.steps, 1))
    roof["fused_ms_per_step"] = fused_ms / args.steps
    roof["fused_share_of_step"] = fused_ms / total_ms if world == 1 else None

    # ---- end to end through the public API with host buffers ----
    e2e = None
    if not args.no_e2e:
        try:
            e2e = run_e2e(torch, B, w, variant, local, world, max(1, min(args.steps, 3)), barrier, args.timeline if rank == 0 else None)
            if measured.get("pcie_d2h_gbs"):
                e2e["pcie_gbs"] = measured["pcie_d2h_gbs"]
                e2e["pcie_h2d_gbs"] = measured["pcie_h2d_gbs"]
                e2e["achieved_d2h_gbs"] = e2e["d2h_bytes_per_step"] / (e2e["ms_per_step"] * 1e-3) / 1e9
                e2e["frac_of_pcie"] = e2e["achieved_d2h_gbs"] / measured["pcie_d2h_gbs"]
        except Exception as ex:                                   # report, never fake
            e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}
    extras = None
    if rank == 0 and world == 1 and not args.no_extras and not args.samples:
        try:
            extras = run_extras(torch, B, w, local, tod)
        except Exception as ex:
            extras = {"error": repr(ex)[:200]}

    variant_name = plan.variant_name
    plan.destroy()
    del tod
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu, _, _ = oracle_sample(w, args.cpu_seconds)
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": workload_config(w, {"variant": variant_name, "parallelism": f"replica x{world}"}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu}
        if extras:
            line["options"] = extras
        if args.samples:
            line["invalid"] = "--samples shrinks the workload: debug only"
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_spaxel_sharded(args, torch, dist, B, W, shard, w, variant, rank, world, local, barrier):
    """Strong scaling over spaxels: rank r simulates spaxels [b_r, e_r) of the SAME observation in
    kelvin (RNG counters keep the global spaxel index), then the common-mode subtraction of Eq. 25: per-rank partial sums
    over [t x chan] (gt_common_mode_partial), ONE all-reduce (NCCL), gt_common_mode_apply on the rank's own slab."""
    dev = f"cuda:{local}"
    b, e = shard.partition_spaxels(w.n_spaxel, world)[rank]
    wk = w.replace(output_unit=1, skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.4)
    r_out = 0.6 * float(np.max(np.hypot(w.daz_rad, w.del_rad))) if w.n_spaxel > 1 else -1.0
    plan = B.Plan(shard.shard_workload(wk, b, e), variant=variant, device=dev)
    tod = torch.empty((w.n_samples, e - b, w.n_chan), dtype=torch.float32, device=dev)
    pwv = torch.empty((w.n_samples, e - b), dtype=torch.float32, device=dev)
    grp = dist if world > 1 else None

    def step():
        plan.simulate(out=tod, pwv_out=pwv)
        acc = torch.stack([pwv.double().sum(), torch.tensor(float(pwv.numel()), dtype=torch.float64, device=dev)])
        if world > 1:
            dist.all_reduce(acc)
        pwv_mean = float((acc[0] / acc[1]).item())                 # the zenith PWV averaged over the observation
        partial, n_out = plan.common_mode_partial(tod, pwv_mean, r_out)
        total, n_tot = shard.common_mode_allreduce(partial, n_out, grp)
        plan.common_mode_apply(tod, pwv_mean, total, n_tot)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local); sampler.start()
    launches0 = plan.launch_count
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record(); e1.synchronize()
    barrier()
    total_ms = shard.max_over_ranks(e0.elapsed_time(e1), grp, device=dev)
    clocks = sampler.stop()
    launches = plan.launch_count - launches0
    name = plan.variant_name
    plan.destroy()
    if rank == 0:
        line = {"metric": METRIC, "value": w.detector_samples() * args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": workload_config(w, {"variant": name, "parallelism": f"spaxel-shard x{world}",
                                              "step": "gt_simulate in kelvin + Eq. 25 common-mode subtraction (per-rank partial sums, "
                                                      "one all-reduce over [t x chan], apply)", "rank0_spaxels": [b, e]}),
                "clocks": clocks, "gpu_launches": int(launches), "e2e": None, "roofline": None, "cpu_baseline": None}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_extras(torch, B, w, local, tod):
    """Device-resident step times of the paper's own options (rows f1-f3), same workload: one warm-up + two timed steps."""
    out = {}
    dev = f"cuda:{local}"
    for name, kw in (("f1_exact_photon_noise_eq17", dict(photon_mode=1)),
                     ("f2_kelvin_output", dict(output_unit=1, skydip_pwv_lo_mm=0.6, skydip_pwv_hi_mm=1.4)),
                     ("f3_timmer_koenig_pink", dict(pink_method=1))):
        t0 = time.perf_counter()
        p = B.Plan(w.replace(**kw), device=dev)
        torch.cuda.synchronize()
        create_ms = 1e3 * (time.perf_counter() - t0)
        p.simulate(out=tod)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(2):
            p.simulate(out=tod)
        e1.record(); e1.synchronize()
        ms = e0.elapsed_time(e1) / 2
        out[name] = {"ms_per_step": ms, "value": w.detector_samples() / (ms * 1e-3), "unit": UNIT, "plan_create_ms": create_ms}
        if name == "f2_kelvin_output" and w.n_spaxel > 1:
            # row f4 on one GPU: the same Kelvin step followed by the common-mode subtraction of Eq. 25-26 (partial sums over
            # the spaxels outside 0.6 of the array radius, then the apply pass); bench.py --shard spaxel is the N > 1 form
            r_out = 0.6 * float(np.max(np.hypot(w.daz_rad, w.del_rad)))

            def cm_step():
                p.simulate(out=tod)
                partial, n_out = p.common_mode_partial(tod, 1.0, r_out)
                p.common_mode_apply(tod, 1.0, partial, n_out)
            cm_step()
            e0.record()
            for _ in range(2):
                cm_step()
            e1.record(); e1.synchronize()
            ms4 = e0.elapsed_time(e1) / 2
            out["f4_kelvin_common_mode"] = {"ms_per_step": ms4, "value": w.detector_samples() / (ms4 * 1e-3), "unit": UNIT}
        p.destroy()
        torch.cuda.empty_cache()
    return out


def run_e2e(torch, B, w, variant, local, world, steps, barrier, timeline=None):
    """Public API from HOST buffers: per step, pinned inputs -> device, gt_plan_create,
    gt_simulate streaming the TOD into pinned host memory, gt_plan_destroy."""
    dev = f"cuda:{local}"
    host = {}
    for name, arr in (("cube", w.cube), ("screen", w.screen), ("atm_lut", w.atm_lut), ("filt", w.filt)):
        if arr is not None:
            host[name] = torch.from_numpy(np.ascontiguousarray(arr, dtype=np.float32)).pin_memory()
    h2d = sum(t.numel() * 4 for t in host.values()) + 16 * w.n_samples
    out = torch.empty((w.n_samples, w.n_spaxel, w.n_chan), dtype=torch.float32, pin_memory=True)
    d2h = out.numel() * 4

    # the workload's large arrays now live in pinned host memory: the binding copies the pinned tensors as they are
    wp = w.replace(**host)

    parts = {"h2d_ms": 0.0, "plan_create_ms": 0.0, "simulate_ms": 0.0, "destroy_ms": 0.0}

    def one(record=None):
        # B.Plan copies the pinned arrays to the device (H2D) and creates the plan; simulate streams to `out`
        t0 = time.perf_counter()
        p = B.Plan(wp, variant=variant, device=dev)
        t1 = time.perf_counter()
        p.simulate(out=out)
        t2 = time.perf_counter()
        if record:
            tl = p.timeline()
            with open(record, "w") as f:
                f.write("# per-chunk device timeline of one end-to-end gt_simulate into pinned host memory (gt_debug_timeline):\n"
                        "# ms after the first chunk's compute begin; compute = geometry + fused + pink kernels on the caller's stream,\n"
                        "# copy = cudaMemcpyAsync D2H of that chunk on the plan's side stream\n"
                        f"# command: python bench.py --steps 1 --warmup 3 --timeline {record}\n"
                        f"# workload: {w.name}, {tl.shape[0]} chunks of {p.chunking()[0]} samples ({p.chunking()[0] * w.n_spaxel * w.n_chan * 4 / 1e6:.0f} MB; the last one is shorter)\n"
                        "# chunk compute_begin compute_end copy_begin copy_end  copy_GB/s  copy_overlaps_next_compute\n")
                chunk_s, row_b = p.chunking()[0], w.n_spaxel * w.n_chan * 4
                for k, r in enumerate(tl):
                    per = min(chunk_s, w.n_samples - k * chunk_s) * row_b
                    ov = "yes" if k + 1 < tl.shape[0] and r[2] < tl[k + 1][1] and r[3] > tl[k + 1][0] else ("-" if k + 1 == tl.shape[0] else "no")
                    f.write(f"{k:4d} {r[0]:9.3f} {r[1]:9.3f} {r[2]:9.3f} {r[3]:9.3f} {per / max(r[3] - r[2], 1e-6) / 1e6:8.1f}  {ov}\n")
                f.write(f"# compute busy {sum(r[1] - r[0] for r in tl):.1f} ms, copy busy {sum(r[3] - r[2] for r in tl):.1f} ms, "
                        f"span {tl[-1][3]:.1f} ms\n")
        p.destroy()
        t3 = time.perf_counter()
        parts["h2d_ms"] += p.upload_ms; parts["plan_create_ms"] += p.create_ms
        parts["simulate_ms"] += 1e3 * (t2 - t1); parts["destroy_ms"] += 1e3 * (t3 - t2)

    one(record=timeline)                                         # warm-up (allocators, pinned pages)
    for k in parts:
        parts[k] = 0.0
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    t = torch.tensor([dt], dtype=torch.float64, device=dev)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dt = float(t.item())
    return {"value": world * w.detector_samples() * steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * dt / steps, "steps": steps,
            "breakdown_ms_per_step": {k: v / steps for k, v in parts.items()},
            "what": "host arrays -> H2D -> gt_plan_create -> gt_simulate into pinned host TOD (chunked D2H on a side stream) -> gt_plan_destroy"}


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
