#!/usr/bin/env python
"""bench.py -- throughput of the Upsilon_Nseg hot path on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W [--workload cfg3] [--n-seg 16] [--impl reference]

A step = one pass of the whole hot path over one batch: tfs_eval (track + Fresnel pixels + gather +
segment sums + combine) over the workload's template bank and tfs_topk of the top 1 %.  The data
grid is uploaded once before timing (SURVEY.md 8(a) row a0 is per dataset, not per batch).
Prints ONE JSON line on rank 0.  N > 1: independent replicas, one per rank.
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

from paper_2510_19047_b200 import synth  # noqa: E402

# Algorithmic bytes per pixel-eval: 8 B complex fp32 datum + 4 B weight
# when the weights are a general per-pixel array; 8 B when they are separable W[a,m,k] = a[m] b[k]
# (tfs_weight_structure 1 or 2: true of every BASELINE.json config), where no per-pixel weight exists to read.
ALG_BYTES_PER_PIXEL_EVAL = {0: 12.0, 1: 8.0, 2: 8.0}
# Algorithmic FMA-pipe lane-slots per window pixel (both channels), far-zone pixel.
# A packed fp32 instruction (FFMA2/FMUL2/FADD2) is one issue slot but two lane-slots of the FMA pipe:
# 10 packed for the two auxiliary-function polynomials (20), h' = Godd(v0) - E Godd(v1) (4 scalar FMA),
# z_A, z_E (4 packed: 8), |h'|^2 and q (1 packed: 2), u + c and u - 1 (2)  ->  36; + 2 MUFU.RCP (own pipe).
ALG_LANE_OPS_PER_PIXEL = 36.0
SM_LANES = 128                       # lane-instructions issued per SM per clock (4 schedulers x 32 lanes)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ---------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# oracle arm (CPU): the dense fp64 oracle, as it stands, on a bounded sample of the workload
# ---------------------------------------------------------------------------------------------
_ORA = {}


def _oracle_one(i):
    from oracle import tfs_oracle as O
    d = _ORA
    r = O.evaluate(d["params"][i:i + 1], d["D"], d["W"], d["gap"], d["grid"], d["N_seg"])
    return float(r["upsilon"][0])


def oracle_throughput(w, coeff, weight, gap, params, N_seg, n_sample, procs):
    """templates/s of oracle/ on `n_sample` templates using `procs` processes (fork; call BEFORE CUDA init)."""
    import multiprocessing as mp
    from oracle import tfs_oracle as O
    c = coeff.astype(np.float64)
    _ORA.update(params=params, D=c[..., 0] + 1j * c[..., 1], W=weight.astype(np.float64), gap=gap,
                grid=O.Grid(w.Nt, w.Nf, w.dt), N_seg=N_seg)
    del c
    idx = list(range(n_sample))
    t0 = time.perf_counter()
    if procs > 1:
        with mp.get_context("fork").Pool(procs) as pool:
            ups = pool.map(_oracle_one, idx, chunksize=1)
    else:
        ups = [_oracle_one(i) for i in idx]
    dt = time.perf_counter() - t0
    _ORA.clear()
    return n_sample / dt, dt, ups


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tfs", choices=["tfs", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(synth.WORKLOADS))
    ap.add_argument("--n-templates", type=int, default=None)
    ap.add_argument("--n-seg", type=int, default=None)
    ap.add_argument("--cpu-sample", type=int, default=None, help="templates timed on the CPU oracle")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--weight-mode", type=int, default=0, choices=[0, 1],
                    help="tfs_opts.weight_mode: 0 = exploit separable weights (default), 1 = general per-pixel path")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    w = synth.WORKLOADS[args.workload]
    n = args.n_templates or w.n_templates
    N_seg = args.n_seg or w.N_seg
    k_top = max(1, n // 100)
    cfg = {"workload": f"{w.name}: Nt={w.Nt} x Nf={w.Nf} x 2 channels (A,E), dt={w.dt:g} s, noise={w.noise}, "
                       f"gaps={w.gaps}, {n} templates, N_seg={N_seg}, top-k k={k_top}",
           "grid_bytes": int(w.Nt * w.Nf * 24), "l2": "inputs larger than L2 (grid 302 MB at cfg3 > 126 MB L2)",
           "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (no collective)"}

    # ---------------- reference arm: the CPU oracle, rank 0 only ----------------
    if args.impl == "reference":
        if rank != 0:
            return 0
        coeff, weight, gap = synth.make_data(w)
        cores = host_cores()
        procs = max(1, min(cores, 16))
        per_step = args.cpu_sample or 4 * procs
        params = synth.make_templates(w, per_step * (args.steps + args.warmup))
        rates = []
        for s in range(args.steps + args.warmup):
            r, dt, _ = oracle_throughput(w, coeff, weight, gap, params[s * per_step:(s + 1) * per_step], N_seg,
                                         per_step, procs)
            if s >= args.warmup:
                rates.append((per_step, dt))
        tot_n = sum(a for a, _ in rates); tot_t = sum(b for _, b in rates)
        val = tot_n / tot_t
        line = {"impl": "reference", "metric": "templates/sec", "value": val, "unit": "templates/s",
                "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * tot_t / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                "cpu_baseline": {"value": val, "unit": "templates/s", "cores": procs, "kind": "oracle",
                                 "sample": f"{per_step} templates of the workload per step (dense fp64 oracle, "
                                           f"{procs} processes)"},
                "e2e": {"value": val, "unit": "templates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # ---------------- our arm ----------------
    coeff, weight, gap = synth.make_data(w)
    params = synth.make_templates(w, n)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = host_cores()
        procs = max(1, min(cores, 16))
        ns = args.cpu_sample or 12 * procs      # ~10-30 s of CPU work at cfg3
        r, dt, ups_cpu = oracle_throughput(w, coeff, weight, gap, params[:ns], N_seg, ns, procs)   # before CUDA init
        cpu_baseline = {"value": r, "unit": "templates/s", "cores": procs, "kind": "oracle",
                        "sample": f"first {ns} templates of the bank, {dt:.1f} s wall (dense fp64 oracle, {procs} "
                                  f"processes of {cores} cores)"}

    import torch
    from paper_2510_19047_b200 import api, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libtfs has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()

    ctx = api.Tfs(w.Nt, w.Nf, w.dt, weight_mode=args.weight_mode)
    ctx.upload_data(coeff, weight, gap)
    d_params = torch.from_numpy(params).to(dev)
    d_ups = torch.empty(n, dtype=torch.float32, device=dev)
    d_idx = torch.empty(k_top, dtype=torch.int64, device=dev)
    d_val = torch.empty(k_top, dtype=torch.float32, device=dev)
    counts = torch.empty(n, dtype=torch.int64, device=dev)
    ctx.count_pixels(d_params, counts)
    torch.cuda.synchronize()
    pixels = int(counts.sum().item())
    pixel_evals = 2 * pixels
    l2_gbs = ctx.probe_l2_bandwidth(32 << 20, 200)
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count

    def step():
        ctx.eval(d_params, N_seg, d_ups)
        ctx.topk(d_ups, k_top, d_idx, d_val)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ctx.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    prof = ctx.get_profile()
    ctx.set_profiling(False)
    clocks = sampler.stop() if rank == 0 else None
    if world > 1:
        t = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps

    # ---------------- e2e: host buffers through the C ABI, copies inside the timed region ----------------
    h_params = torch.from_numpy(params).pin_memory()
    h_ups = torch.empty(n, dtype=torch.float32).pin_memory()
    h_idx = torch.empty(k_top, dtype=torch.int64).pin_memory()
    h_val = torch.empty(k_top, dtype=torch.float32).pin_memory()

    def step_e2e():
        ctx.eval(h_params.numpy(), N_seg, h_ups.numpy())
        ctx.topk(h_ups.numpy(), k_top, h_idx.numpy(), h_val.numpy())

    step_e2e()
    barrier()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e2.record()
    for _ in range(args.steps):
        step_e2e()
    e3.record()
    barrier()
    wall_e2e = time.perf_counter() - t0
    ms_e2e = max(e2.elapsed_time(e3), 1e3 * wall_e2e) / args.steps
    if world > 1:
        t = torch.tensor([ms_e2e], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_e2e = float(t.item())
    same = bool(np.array_equal(h_ups.numpy(), d_ups.cpu().numpy()))

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = measured_peaks()
    n_launch = max(prof["main_kernel_launches"], 1)
    kern_ms = prof["main_kernel_ms"] / n_launch                    # per main-kernel launch
    launches_per_step = n_launch / args.steps
    wstruct = ctx.weight_structure()
    bytes_per_launch = ALG_BYTES_PER_PIXEL_EVAL[wstruct] * pixel_evals / launches_per_step
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    # roofline terms: the gathers are served by the L2 (tile-major order), so the
    # byte term is quoted against the L2 read bandwidth probed in this run; the HBM figure is given for
    # context (what the same bytes would cost if every gather missed the L2); the ALU term is the
    # algorithmic instruction count against the issue rate at the clock seen during the timed region.
    sm_mhz = (clocks or {}).get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
    alu_peak = sm_count * SM_LANES * sm_mhz * 1e6 / 1e12           # T lane-instructions / s
    alu_ach = ALG_LANE_OPS_PER_PIXEL * pixels / launches_per_step / (kern_ms * 1e-3) / 1e12
    terms = {
        "l2": {"achieved": achieved, "peak": l2_gbs, "unit": "GB/s", "frac": achieved / l2_gbs,
               "peak_source": "tfs_probe_l2_bandwidth, 32 MiB buffer, this run"},
        "hbm_if_every_gather_missed_l2": {"achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                          "frac": achieved / peaks["hbm_gbs"], "peak_source": peak_src},
        "alu": {"achieved": alu_ach, "peak": alu_peak, "unit": "T lane-instr/s", "frac": alu_ach / alu_peak,
                "peak_source": f"{sm_count} SMs x {SM_LANES} lanes x {sm_mhz:.0f} MHz (sampled)"},
    }
    bound = "l2" if terms["l2"]["frac"] >= terms["alu"]["frac"] else "alu"
    line = {
        "metric": "templates/sec", "value": world * n / (ms_step * 1e-3), "unit": "templates/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": cfg,
        "pixel_evals_per_sec": world * pixel_evals / (ms_step * 1e-3),
        "pixel_evals_per_template": pixel_evals / n,
        "roofline": {"bound": bound, "kernel": "eval_tiles_kernel", "achieved": terms[bound]["achieved"],
                     "peak": terms[bound]["peak"], "peak_source": terms[bound]["peak_source"],
                     "unit": terms[bound]["unit"], "frac": terms[bound]["frac"], "traffic": None,
                     "algorithmic_bytes_per_launch": bytes_per_launch,
                     "algorithmic_bytes_per_pixel_eval": ALG_BYTES_PER_PIXEL_EVAL[wstruct],
                     "weight_structure": wstruct, "kernel_ms_per_launch": kern_ms,
                     "kernel_share_of_step": prof["main_kernel_ms"] / ms_total, "terms": terms},
        "cpu_baseline": cpu_baseline,
        "e2e": {"value": world * n / (ms_e2e * 1e-3), "unit": "templates/s",
                "h2d_bytes_per_step": int(params.nbytes + h_ups.numpy().nbytes),
                "d2h_bytes_per_step": int(h_ups.numpy().nbytes + h_idx.numpy().nbytes + h_val.numpy().nbytes),
                "ms_per_step": ms_e2e, "matches_device_path": same},
        "gpu_launches": int(prof["kernel_launches"]),
        "clocks": clocks,
    }
    extra = os.path.join(ROOT, "profiles", "roofline_traffic.json")      # ncu-derived, committed by hand
    if os.path.exists(extra):
        try:
            line["roofline"].update(json.load(open(extra)).get(w.name, {}))
        except Exception:
            pass
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
