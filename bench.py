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

from paper_2510_19047_b200 import replicas, synth  # noqa: E402

# Algorithmic bytes per pixel-eval: 8 B complex fp32 datum + 4 B weight
# when the weights are a general per-pixel array; 8 B when they are separable W[a,m,k] = a[m] b[k]
# (tfs_weight_structure 1 or 2: true of every BASELINE.json config), where no per-pixel weight exists to read.
ALG_BYTES_PER_PIXEL_EVAL = {0: 12.0, 1: 8.0, 2: 8.0}
# Algorithmic FMA-pipe lane-slots per window pixel (both channels), far-zone pixel.
# A packed fp32 instruction (FFMA2/FMUL2/FADD2) is one issue slot but two lane-slots of the FMA pipe:
# 10 packed for the two auxiliary-function polynomials (20), h' = Godd(v0) - E Godd(v1) (4 scalar FMA),
# z_A, z_E (4 packed: 8), |h'|^2 and q (1 packed: 2), u + c and u - 1 (2)  ->  36; + 2 MUFU.RCP (own pipe).
ALG_LANE_OPS_PER_PIXEL = 36.0
# The kernels evaluate a window offset in one of three tiers, chosen per warp (tfs_kernels.cuh); counted by the same rule:
#   FAR  36 (above);  FAR2 24 (leading asymptotic term: 4 packed instead of 10 for f, g);
#   NEAR 28 (table: v0, v1 (2), two look-ups = 1 + |v|, index FMA, packed interpolation (8), sign/scale of Godd (4),
#            h' (4), z_A, z_E (8), q (2); the branch for pixels inside the swept band and the slow-chirp series are extra)
TIER_LANE_OPS = {"far2": 24.0, "far": 36.0, "near": 28.0}
SM_LANES = 128                       # lane-instructions issued per SM per clock (4 schedulers x 32 lanes)
SMEM_BYTES_PER_CLK = 128             # shared-memory bandwidth per SM per clock (B300_MICROARCH.md: 128/N B/clk/SM)


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
    return float(r["upsilon"][0]), int((r["seg_hh"][0] > 0).sum())


def _sparse_eval(p, g, o, seg, coeff, weight, gap, N_seg):
    """Upsilon of one template from its window pixels only, with the oracle's track, kernel and combine routines."""
    from oracle import tfs_oracle as O
    tr = O.track(p[0], p[1], p[2], p[7], g, o, gap)
    ms = np.nonzero(tr["active"])[0]
    z = np.zeros(N_seg, dtype=np.complex128)
    hh = np.zeros(N_seg)
    if ms.size:
        lo, hi = tr["k_lo"][ms], tr["k_hi"][ms]
        mm = np.repeat(ms, hi - lo + 1)
        kk = np.concatenate([np.arange(a, b + 1) for a, b in zip(lo, hi)])
        H = O.kernel_pixels(tr["x"][mm], tr["c"][mm], tr["phi"][mm], tr["A"][mm], kk)
        T = (p[3] + 1j * p[4], p[5] + 1j * p[6])
        for a in range(2):
            D = coeff[a, mm, kk, 0].astype(np.float64) + 1j * coeff[a, mm, kk, 1]
            Wp = weight[a, mm, kk].astype(np.float64)
            z += T[a] * (np.bincount(seg[mm], weights=(Wp * np.conj(D) * H).real, minlength=N_seg) +
                         1j * np.bincount(seg[mm], weights=(Wp * np.conj(D) * H).imag, minlength=N_seg))
            hh += abs(T[a]) ** 2 * np.bincount(seg[mm], weights=Wp * np.abs(H) ** 2, minlength=N_seg)
    return float(O.combine(z, hh)[1])


def sparse_cpu_rate(w, coeff, weight, gap, params, N_seg, budget_s=6.0):
    """The analogue of the paper's single-core CPU curve (Fig. 1): the same statistic evaluated
    on the track's window pixels only, one template at a time on ONE core, with the oracle's own track,
    kernel and combine routines (numpy fp64) -- a labelled second CPU line, not the oracle (which sums
    over every pixel).  Returns (templates/s, templates timed)."""
    from oracle import tfs_oracle as O
    g = O.Grid(w.Nt, w.Nf, w.dt)
    o = O.Opts()
    seg = O.segment_of_bin(np.arange(w.Nt), w.Nt, N_seg)
    t0 = time.perf_counter()
    done = 0
    for p in params:
        _sparse_eval(p, g, o, seg, coeff, weight, gap, N_seg)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    return done / (time.perf_counter() - t0), done


def _sparse_one(i):
    d = _ORA
    return _sparse_eval(d["params"][i], d["grid"], d["opts"], d["seg"], d["coeff"], d["weight"], d["gap"], d["N_seg"])


def sparse_cpu_rate_mp(w, coeff, weight, gap, params, N_seg, procs):
    """The window-sparse CPU evaluation on `procs` processes (fork; call BEFORE CUDA init): the fairest CPU line this
    bench prints -- what a multi-core CPU implementation that, like the GPU path, touches the window pixels only would
    reach with numpy.  Returns (templates/s, seconds, [Upsilon])."""
    import multiprocessing as mp
    from oracle import tfs_oracle as O
    _ORA.update(params=params, coeff=coeff, weight=weight, gap=gap, grid=O.Grid(w.Nt, w.Nf, w.dt), opts=O.Opts(),
                seg=O.segment_of_bin(np.arange(w.Nt), w.Nt, N_seg), N_seg=N_seg)
    idx = list(range(len(params)))
    t0 = time.perf_counter()
    if procs > 1:
        with mp.get_context("fork").Pool(procs) as pool:
            ups = pool.map(_sparse_one, idx, chunksize=max(1, len(idx) // (8 * procs)))
    else:
        ups = [_sparse_one(i) for i in idx]
    dt = time.perf_counter() - t0
    _ORA.clear()
    return len(idx) / dt, dt, ups


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


def time_leg(api, torch, ctx, w, d_params, n, N_seg, k_top, steps, warmup, info, dev, sample_clocks):
    """Device-timed leg: `warmup` untimed steps, then exactly `steps` steps bracketed by barrier + synchronize.
    Returns dict(ms_step, prof, clocks, d_ups)."""
    d_ups = torch.empty(n, dtype=torch.float32, device=dev)
    d_idx = torch.empty(k_top, dtype=torch.int64, device=dev)
    d_val = torch.empty(k_top, dtype=torch.float32, device=dev)

    def step():
        ctx.eval(d_params, N_seg, d_ups)
        ctx.topk(d_ups, k_top, d_idx, d_val)

    def barrier():
        replicas.barrier(info)
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    sampler = ClockSampler(info.local_rank)
    if sample_clocks:
        sampler.start()
    ctx.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    prof = ctx.get_profile_kernels()
    ctx.set_profiling(False)
    clocks = sampler.stop() if sample_clocks else None
    ms_total = replicas.max_over_ranks(ms_total, info, dev)
    return dict(ms_step=ms_total / steps, ms_total=ms_total, prof=prof, clocks=clocks, d_ups=d_ups, d_idx=d_idx, d_val=d_val)


def tier_census(ctx, step):
    """One untimed step with the library's tier counters on: pixel slots evaluated per tier (tfs_tier_census)."""
    import torch
    ctx.tier_census(True)
    step()
    torch.cuda.synchronize()
    c = ctx.tier_census(False)
    slots = {"far2": c[0], "far": c[1] + c[3], "near": c[2] + c[4]}
    total = max(sum(slots.values()), 1)
    mean_ops = sum(TIER_LANE_OPS[k] * v for k, v in slots.items()) / total
    return {"pixel_slots": slots, "slab_kernel": {"far2": c[0], "far": c[1], "near": c[2]},
            "list_kernel": {"far": c[3], "near": c[4]}, "lane_ops_per_tier": TIER_LANE_OPS,
            "mean_lane_ops_per_slot": mean_ops, "pixel_slots_total": total}


def roofline_terms(leg, steps, pixels, wstruct, l2_gbs, peaks, peak_src, sm_count, sm_mhz, census=None, issue=None):
    """The roofline terms of the evaluation kernels (eval_list_kernel + eval_slab_kernel, one pair per step)."""
    n_launch = max(leg["prof"]["eval_launches"], 1)
    kern_ms = (leg["prof"]["slab_kernel_ms"] + leg["prof"]["list_kernel_ms"]) / n_launch
    per_step = n_launch / steps
    bytes_per_launch = ALG_BYTES_PER_PIXEL_EVAL[wstruct] * 2 * pixels / per_step
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    smem_peak = sm_count * SMEM_BYTES_PER_CLK * sm_mhz * 1e6 / 1e9
    alu_peak = sm_count * SM_LANES * sm_mhz * 1e6 / 1e12           # T lane-instructions / s
    # arithmetic actually needed: the tiers the kernels executed (census), on the window pixels only (the padding slots
    # of inactive lanes and masked tails are waste, not work); without a census the flat far-tier figure
    ops = census["mean_lane_ops_per_slot"] if census else ALG_LANE_OPS_PER_PIXEL
    alu_ach = ops * pixels / per_step / (kern_ms * 1e-3) / 1e12
    alu_flat = ALG_LANE_OPS_PER_PIXEL * pixels / per_step / (kern_ms * 1e-3) / 1e12
    terms = {
        "l2": {"achieved": achieved, "peak": l2_gbs, "unit": "GB/s", "frac": achieved / l2_gbs,
               "peak_source": "tfs_probe_l2_bandwidth, 32 MiB buffer, this run (the SM's L1 -> register return path)"},
        "smem": {"achieved": achieved, "peak": smem_peak, "unit": "GB/s", "frac": achieved / smem_peak,
                 "peak_source": f"{sm_count} SMs x {SMEM_BYTES_PER_CLK} B/clk x {sm_mhz:.0f} MHz (sampled): where the slab "
                                "kernel's gathers are served"},
        "hbm_if_every_gather_missed_l2": {"achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                          "frac": achieved / peaks["hbm_gbs"], "peak_source": peak_src},
        "alu": {"achieved": alu_ach, "peak": alu_peak, "unit": "T lane-instr/s", "frac": alu_ach / alu_peak,
                "peak_source": f"{sm_count} SMs x {SM_LANES} lanes x {sm_mhz:.0f} MHz (sampled)",
                "lane_ops_per_pixel": ops,
                "lane_ops_source": "tier census of this run (tfs_tier_census)" if census else "flat far-tier count",
                "frac_flat_36_ops": alu_flat / alu_peak},
    }
    if census:
        terms["alu"]["tier_census"] = census
        terms["alu"]["padding_slots_frac"] = 1.0 - pixels / census["pixel_slots_total"]      # the census covers one whole step
    if issue:
        lanes = max(32.0 * issue[0], 64.0 * issue[1])
        meas_peak = sm_count * lanes * sm_mhz * 1e6 / 1e12
        terms["alu"].update({"peak_measured": meas_peak, "frac_of_measured_peak": alu_ach / meas_peak,
                             "peak_measured_source": f"tfs_probe_fp32_issue, this run: {issue[0]:.2f} scalar FFMA / "
                                                     f"{issue[1]:.2f} packed FFMA2 warp-instr/clk/SM = {lanes:.1f} "
                                                     "FMA lane-slots/clk/SM"})
    return terms, kern_ms, bytes_per_launch


def _wdm_oracle_one(i):
    from oracle import tfs_wdm as Wd
    d = _ORA
    r = Wd.evaluate(d["params"][i:i + 1], d["D"], d["W"], d["gap"], d["grid"], d["N_seg"])
    return float(r["upsilon"][0]), int((r["seg_gram"][0, :, 0] > 0).sum())


def main_wdm(args, info, w, n, N_seg, k_top, cfg):
    """The same step in the WDM wavelet pixel basis (tfs_opts.basis = 1): real coefficients on the same Nt x Nf
    grid (pixel duration Nf dt), general per-pixel weights.  One timed leg + the oracle (oracle/tfs_wdm.py) on a
    bounded sample; algorithmic bytes per pixel-eval: 4 B datum + 4 B weight."""
    import multiprocessing as mp
    rank, world = info.rank, info.world
    if args.impl == "reference" and rank != 0:
        return 0                                   # the reference arm runs on rank 0 alone
    cfg = dict(cfg, workload=cfg["workload"].replace("x 2 channels (A,E)", "x 2 channels (A,E), real WDM wavelet pixels (basis = 1)"))
    coeff_c, weight, gap = synth.make_data(w)
    coeff = np.ascontiguousarray(coeff_c[..., 0])                        # real pixels with the same noise model
    del coeff_c
    params = synth.make_templates(w, n, seed=replicas.bank_seed(w.seed, rank))
    if args.impl == "reference" or (rank == 0 and world == 1 and not args.no_cpu_baseline):
        from oracle import tfs_wdm as Wd
        cores = host_cores()
        procs = max(1, min(cores, 16))
        ns = args.cpu_sample or 4 * procs
        _ORA.update(params=params, D=coeff.astype(np.float64), W=weight.astype(np.float64), gap=gap,
                    grid=Wd.WdmGrid(w.Nt, w.Nf, w.dt), N_seg=N_seg)
        t0 = time.perf_counter()
        with mp.get_context("fork").Pool(procs) as pool:
            ora = pool.map(_wdm_oracle_one, list(range(ns)), chunksize=1)
        dt = time.perf_counter() - t0
        _ORA.clear()
        cpu_baseline = {"value": ns / dt, "unit": "templates/s", "cores": procs, "kind": "oracle",
                        "sample": f"first {ns} templates of the bank, {dt:.1f} s wall (oracle/tfs_wdm.py, {procs} processes)"}
        if args.impl == "reference":
            if rank == 0:
                print(json.dumps({"impl": "reference", "metric": "templates/sec", "value": ns / dt, "unit": "templates/s",
                                  "n_gpus": args.gpus, "steps": 1, "warmup": 0, "ms_per_step": 1e3 * dt,
                                  "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                                  "data": "synthetic", "config": cfg, "cpu_baseline": cpu_baseline,
                                  "e2e": {"value": ns / dt, "unit": "templates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                                  "gpu_launches": 0}))
            return 0
    else:
        cpu_baseline, ora = None, None
    import torch
    from paper_2510_19047_b200 import api, build
    torch.cuda.set_device(info.local_rank)
    dev = torch.device("cuda", info.local_rank)
    replicas.init(info, "nccl", dev)
    if rank == 0:
        build.build()
    replicas.barrier(info)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, basis=1)
    ctx.upload_data(coeff, weight, gap)
    d_params = torch.from_numpy(params).to(dev)
    counts = torch.empty(n, dtype=torch.int64, device=dev)
    ctx.count_pixels(d_params, counts)
    torch.cuda.synchronize()
    pixels = int(counts.sum().item())
    l2_gbs = ctx.probe_l2_bandwidth(32 << 20, 200)
    warm = max(args.warmup, 3)
    leg = time_leg(api, torch, ctx, w, d_params, n, N_seg, k_top, args.steps, warm, info, dev, rank == 0)
    parity = None
    if ora is not None:
        uo = np.array([u for u, _ in ora]); neff = np.maximum(np.array([e for _, e in ora]), 1)
        err = np.abs(leg["d_ups"][:len(uo)].cpu().numpy().astype(np.float64) - uo) / np.maximum(uo, 2.0 * neff)
        parity = {"n": int(len(uo)), "max_norm_err": float(err.max()), "tolerance": 1e-4, "ok": bool(err.max() <= 1e-4),
                  "criterion": "|dUpsilon| <= 1e-4 max(Upsilon, 2 N_eff), GPU output of the timed run vs oracle/tfs_wdm.py"}
    h_params = torch.from_numpy(params).pin_memory()
    h_ups = torch.empty(n, dtype=torch.float32).pin_memory()
    h_idx = torch.empty(k_top, dtype=torch.int64).pin_memory()
    h_val = torch.empty(k_top, dtype=torch.float32).pin_memory()
    ctx.eval(h_params.numpy(), N_seg, h_ups.numpy())
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.eval(h_params.numpy(), N_seg, h_ups.numpy())
        ctx.topk(h_ups.numpy(), k_top, h_idx.numpy(), h_val.numpy())
    torch.cuda.synchronize()
    ms_e2e = replicas.max_over_ranks(1e3 * (time.perf_counter() - t0) / args.steps, info, dev)
    if rank != 0:
        replicas.finish(info)
        return 0
    prof = leg["prof"]
    n_launch = max(prof["eval_launches"], 1)
    kern_ms = (prof["slab_kernel_ms"] + prof["list_kernel_ms"]) / n_launch
    bytes_per_launch = 8.0 * 2 * pixels / (n_launch / args.steps)
    achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
    line = {"metric": "templates/sec", "value": replicas.aggregate_rate(n, leg["ms_step"] * 1e-3, info), "unit": "templates/s", "n_gpus": world,
            "steps": args.steps, "warmup": warm, "ms_per_step": leg["ms_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfg,
            "pixel_evals_per_sec": world * 2 * pixels / (leg["ms_step"] * 1e-3), "pixel_evals_per_template": 2 * pixels / n,
            "roofline": {"bound": "l2", "kernel": "eval_wdm_kernel", "achieved": achieved, "peak": l2_gbs, "unit": "GB/s",
                         "frac": achieved / l2_gbs, "traffic": None,
                         "peak_source": "tfs_probe_l2_bandwidth, 32 MiB buffer, this run",
                         "algorithmic_bytes_per_pixel_eval": 8.0, "algorithmic_bytes_per_launch": bytes_per_launch,
                         "kernel_ms_per_launch": kern_ms,
                         "note": "a first kernel for this basis: four table look-ups and two fp64 phase reductions per pixel; "
                                 "it is instruction-bound, far from the byte roof"},
            "cpu_baseline": cpu_baseline, "parity": parity,
            "e2e": {"value": replicas.aggregate_rate(n, ms_e2e * 1e-3, info), "unit": "templates/s", "h2d_bytes_per_step": int(params.nbytes),
                    "d2h_bytes_per_step": int(4 * n + 12 * k_top), "ms_per_step": ms_e2e},
            "gpu_launches": int(prof["kernel_launches"]), "clocks": leg["clocks"]}
    print(json.dumps(line))
    replicas.finish(info)
    return 0


# ---------------------------------------------------------------------------------------------
# secondary legs of the default run: the configurations next to the headline one, each timed on the device for a
# few steps and compared with the oracle on SEC_ROWS rows of its own bank (so that they are driver-witnessed numbers)
# ---------------------------------------------------------------------------------------------
SEC_ROWS = 64
SEC_KNOTS, SEC_F0, SEC_STEP = 16, 1e-3, 6.6e-3          # transfer tables: 16 knots over 1-100 mHz


def _sec_one(job):
    leg, i = job
    d = _ORA[leg]
    from oracle import tfs_oracle as O
    p = d["params"][i:i + 1]
    if leg == "aet_tables":
        r = O.evaluate_tf(p, d["tables"][i:i + 1], SEC_F0, SEC_STEP, d["D"], d["W"], d["gap"], d["grid"], d["N_seg"])
    elif leg == "wdm":
        from oracle import tfs_wdm as Wd
        r = Wd.evaluate(p, d["D"], d["W"], d["gap"], d["grid"], d["N_seg"])
        return float(r["upsilon"][0]), int((r["seg_gram"][0, :, 0] > 0).sum())
    else:
        r = O.evaluate(p, d["D"], d["W"], d["gap"], d["grid"], d["N_seg"], d["opts"])
    return float(r["upsilon"][0]), int((r["seg_hh"][0] > 0).sum())


def secondary_inputs(w, coeff, weight, gap):
    """Seeded inputs of the four secondary legs (host arrays; no method arithmetic)."""
    rng = np.random.default_rng(33)
    n_aet, n_tuk, n_wdm = 200_000, 100_000, 500_000
    w4 = synth.WORKLOADS["cfg4"]
    c4, wt4, g4 = synth.make_data(w4)
    return {
        "aet_tables": dict(what="A, E, T (third channel = a copy of A's data) with a 16-knot complex transfer table per template "
                                "and channel interpolated per tranche (tfs_eval_tf), cfg3 grid and bank",
                           coeff=np.ascontiguousarray(np.concatenate([coeff, coeff[:1]])),
                           weight=np.ascontiguousarray(np.concatenate([weight, weight[:1]])), gap=gap, w=w, N_seg=w.N_seg,
                           params=synth.make_templates(w, n_aet),
                           tables=rng.standard_normal((n_aet, 3, SEC_KNOTS, 2)).astype(np.float32)),
        "tukey_0.1": dict(what="window-aware template, tukey_alpha = 0.1 (P:271), cfg3 grid and bank", coeff=coeff, weight=weight,
                          gap=gap, w=w, N_seg=w.N_seg, params=synth.make_templates(w, n_tuk)),
        "cfg4": dict(what="BASELINE.json configs[3]: one batch of 2^20 templates (20 % merging inside the grid), N_seg = 32",
                     coeff=c4, weight=wt4, gap=g4, w=w4, N_seg=w4.N_seg, params=synth.make_templates(w4, w4.n_templates)),
        "wdm": dict(what="real WDM wavelet pixels (tfs_opts.basis = 1) on the cfg3-shaped grid, general per-pixel weights",
                    coeff=np.ascontiguousarray(coeff[..., 0]), weight=weight, gap=gap, w=w, N_seg=w.N_seg,
                    params=synth.make_templates(w, n_wdm)),
    }


def secondary_oracle(sec, procs):
    """Oracle Upsilon of the first SEC_ROWS rows of every secondary leg (fork pool: call BEFORE CUDA init)."""
    import multiprocessing as mp
    from oracle import tfs_oracle as O
    from oracle import tfs_wdm as Wd
    for leg, d in sec.items():
        w = d["w"]
        if leg == "wdm":
            _ORA[leg] = dict(params=d["params"], D=d["coeff"].astype(np.float64), W=d["weight"].astype(np.float64), gap=d["gap"],
                             grid=Wd.WdmGrid(w.Nt, w.Nf, w.dt), N_seg=d["N_seg"])
            continue
        c = d["coeff"].astype(np.float64)
        _ORA[leg] = dict(params=d["params"], D=c[..., 0] + 1j * c[..., 1], W=d["weight"].astype(np.float64), gap=d["gap"],
                         grid=O.Grid(w.Nt, w.Nf, w.dt), N_seg=d["N_seg"],
                         opts=O.Opts(tukey_alpha=0.1) if leg == "tukey_0.1" else O.Opts())
        if leg == "aet_tables":
            t = d["tables"][:SEC_ROWS].astype(np.float64)
            _ORA[leg]["tables"] = t[..., 0] + 1j * t[..., 1]
    jobs = [(leg, i) for leg in sec for i in range(SEC_ROWS)]
    t0 = time.perf_counter()
    with mp.get_context("fork").Pool(procs) as pool:
        out = pool.map(_sec_one, jobs, chunksize=1)
    dt = time.perf_counter() - t0
    _ORA.clear()
    res = {leg: out[j * SEC_ROWS:(j + 1) * SEC_ROWS] for j, leg in enumerate(sec)}
    return res, dt


def secondary_legs(api, torch, dev, sec, ora, steps=3):
    """Device-timed secondary legs (CUDA events around `steps` calls after two warm-up calls) + parity with `ora`."""
    out = {}
    for leg, d in sec.items():
        w, N_seg = d["w"], d["N_seg"]
        kw = {"aet_tables": dict(n_channels=3), "tukey_0.1": dict(tukey_alpha=0.1), "wdm": dict(basis=1)}.get(leg, {})
        ctx = api.Tfs(w.Nt, w.Nf, w.dt, **kw)
        ctx.upload_data(d["coeff"], d["weight"], d["gap"])
        dp = torch.from_numpy(d["params"]).to(dev)
        n = dp.shape[0]
        ups = torch.empty(n, dtype=torch.float32, device=dev)
        counts = torch.empty(n, dtype=torch.int64, device=dev)
        ctx.count_pixels(dp, counts)
        if leg == "aet_tables":
            tab = torch.from_numpy(d["tables"]).to(dev)
            call = lambda: ctx.eval_tf(dp, N_seg, tab, SEC_KNOTS, SEC_F0, SEC_STEP, ups)
        else:
            call = lambda: ctx.eval(dp, N_seg, ups)
        for _ in range(2):
            call()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            call()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        n_ch = 3 if leg == "aet_tables" else 2
        r = {"what": d["what"], "templates": int(n), "N_seg": int(N_seg), "ms_per_call": ms, "value": n / (ms * 1e-3),
             "unit": "templates/s", "pixel_evals_per_sec": n_ch * int(counts.sum().item()) / (ms * 1e-3), "steps": steps}
        if ora is not None:
            uo = np.array([u for u, _ in ora[leg]]); neff = np.maximum(np.array([e for _, e in ora[leg]]), 1)
            err = np.abs(ups[:len(uo)].cpu().numpy().astype(np.float64) - uo) / np.maximum(uo, 2.0 * neff)
            r["parity"] = {"n": int(len(uo)), "max_norm_err": float(err.max()), "tolerance": 1e-4, "ok": bool(err.max() <= 1e-4),
                           "n_active": int((uo > 0).sum())}
        out[leg] = r
        ctx.destroy()
        del dp, ups, counts
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the secondary legs (A,E,T + tables, window-aware template, cfg4, WDM basis)")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tfs", choices=["tfs", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(synth.WORKLOADS))
    ap.add_argument("--n-templates", type=int, default=None)
    ap.add_argument("--n-seg", type=int, default=None)
    ap.add_argument("--cpu-sample", type=int, default=None, help="templates timed on the CPU oracle")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-general-leg", action="store_true",
                    help="skip the second timed leg with general per-pixel weights (weight_mode = 1)")
    ap.add_argument("--basis", default="sft", choices=["sft", "wdm"],
                    help="sft: the paper's complex short-time Fourier tranches (headline); wdm: real WDM wavelet pixels "
                         "(tfs_opts.basis = 1, SURVEY.md 8(f) NEXT-1) on the same grid shape")
    ap.add_argument("--weight-mode", type=int, default=0, choices=[0, 1],
                    help="tfs_opts.weight_mode of the headline leg: 0 = exploit separable weights (default), 1 = general per-pixel path")
    args = ap.parse_args()

    info = replicas.RankInfo.from_env()
    rank, world, local_rank = info.rank, info.world, info.local_rank

    w = synth.WORKLOADS[args.workload]
    n = args.n_templates or w.n_templates
    N_seg = args.n_seg or w.N_seg
    k_top = max(1, n // 100)
    grid_bytes = int(w.Nt * w.Nf * 24)
    cfg = {"workload": f"{w.name}: Nt={w.Nt} x Nf={w.Nf} x 2 channels (A,E), dt={w.dt:g} s, noise={w.noise}, "
                       f"gaps={w.gaps}, {n} templates, N_seg={N_seg}, top-k k={k_top}",
           "grid_bytes": grid_bytes,
           "l2": (f"inputs larger than L2 (grid {grid_bytes / 1e6:.0f} MB + {n * 64 / 1e6:.0f} MB of parameters + the step's "
                  "partials/lists > 126 MB L2)" if grid_bytes + n * 64 > 126e6 else
                  f"inputs fit the L2 (grid {grid_bytes / 1e6:.0f} MB): the step's own scratch (partials, item lists) is rewritten "
                  "every step"),
           "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (no collective), one seeded bank per rank"}

    if args.basis == "wdm":
        return main_wdm(args, info, w, n, N_seg, k_top, cfg)

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
    # every rank its own seeded bank (rank 0 = the 1-GPU bank)
    params = synth.make_templates(w, n, seed=replicas.bank_seed(w.seed, rank))

    cpu_baseline = None
    ora = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = host_cores()
        procs = max(1, min(cores, 16))
        ns = args.cpu_sample or 64 * procs      # ~60 s of CPU work at cfg3 on 16 cores (why not 4096)
        r, dt, ora = oracle_throughput(w, coeff, weight, gap, params[:ns], N_seg, ns, procs)   # before CUDA init
        sp_rate, sp_n = sparse_cpu_rate(w, coeff, weight, gap, params[:ns], N_seg)
        mp_rate, mp_dt, mp_ups = sparse_cpu_rate_mp(w, coeff, weight, gap, params[:ns], N_seg, procs)
        dense_ups = np.array([u for u, _ in ora])
        mp_err = float(np.max(np.abs(np.array(mp_ups) - dense_ups) / np.maximum(dense_ups, 2.0 * N_seg)))
        cpu_baseline = {"value": r, "unit": "templates/s", "cores": procs, "kind": "oracle",
                        "sample": f"first {ns} templates of the bank, {dt:.1f} s wall (dense fp64 oracle, {procs} "
                                  f"processes of {cores} cores)",
                        "sparse_single_core": {"value": sp_rate, "unit": "templates/s", "cores": 1, "templates": sp_n,
                                               "what": "window pixels only, one template at a time with the oracle's "
                                                       "track/kernel routines (analogue of the paper's Fig. 1 CPU "
                                                       "curve, P:243); not the oracle"},
                        "sparse_multi_core": {"value": mp_rate, "unit": "templates/s", "cores": procs, "templates": ns,
                                              "seconds": mp_dt, "max_err_vs_dense_oracle": mp_err,
                                              "what": "the same window-sparse evaluation on all the processes the dense "
                                                      "oracle used, checked against the dense oracle's Upsilon on every "
                                                      "template of the sample: the CPU figure to compare the GPU arm "
                                                      "with (the dense oracle above sums over every pixel of the grid "
                                                      "and is slow by construction)"}}

    sec, sec_ora, sec_dt, sec_err = None, None, None, None
    if rank == 0 and world == 1 and not args.no_secondary and w.name == "cfg3":
        try:        # the secondary legs must never take the headline measurement down with them
            sec = secondary_inputs(w, coeff, weight, gap)
            if not args.no_cpu_baseline:
                sec_ora, sec_dt = secondary_oracle(sec, max(1, min(host_cores(), 16)))      # before CUDA init (fork)
        except Exception as exc:
            sec, sec_ora, sec_err = None, None, f"{type(exc).__name__}: {exc}"

    import torch
    from paper_2510_19047_b200 import api, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libtfs has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    replicas.init(info, "nccl", dev)
    if rank == 0:
        build.build()
    replicas.barrier(info)

    ctx = api.Tfs(w.Nt, w.Nf, w.dt, weight_mode=args.weight_mode)
    ctx.upload_data(coeff, weight, gap)
    d_params = torch.from_numpy(params).to(dev)
    counts = torch.empty(n, dtype=torch.int64, device=dev)
    ctx.count_pixels(d_params, counts)
    torch.cuda.synchronize()
    pixels = int(counts.sum().item())
    pixel_evals = 2 * pixels
    # active-pixel histogram of the bank (templates that start above the band or merge at once are empty)
    cq = counts.cpu().numpy()
    pix_hist = {"zero_frac": float((cq == 0).mean()),
                "quantiles_pixels_per_template": {q: int(np.quantile(cq, float(q))) for q in ("0.10", "0.25", "0.50", "0.75", "0.90", "1.00")}}
    l2_gbs = ctx.probe_l2_bandwidth(32 << 20, 200)
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    warm = max(args.warmup, 3)

    leg = time_leg(api, torch, ctx, w, d_params, n, N_seg, k_top, args.steps, warm, info, dev, rank == 0)
    ms_step, clocks, d_ups = leg["ms_step"], leg["clocks"], leg["d_ups"]

    # ---------------- parity of the timed output with the oracle values computed above ----------------
    parity = None
    if ora is not None:
        uo = np.array([u for u, _ in ora])
        neff = np.maximum(np.array([e for _, e in ora]), 1)
        ug = d_ups[:len(uo)].cpu().numpy().astype(np.float64)
        err = np.abs(ug - uo) / np.maximum(uo, 2.0 * neff)
        parity = {"n": int(len(uo)), "max_norm_err": float(err.max()), "tolerance": 1e-4,
                  "criterion": "C12: |dUpsilon| <= 1e-4 max(Upsilon, 2 N_eff), GPU output of the timed run vs oracle/",
                  "ok": bool(err.max() <= 1e-4)}

    # ---------------- e2e: host buffers through the C ABI, copies inside the timed region ----------------
    h_params = torch.from_numpy(params).pin_memory()
    h_ups = torch.empty(n, dtype=torch.float32).pin_memory()
    h_idx = torch.empty(k_top, dtype=torch.int64).pin_memory()
    h_val = torch.empty(k_top, dtype=torch.float32).pin_memory()

    def step_e2e():
        ctx.eval(h_params.numpy(), N_seg, h_ups.numpy())
        ctx.topk(h_ups.numpy(), k_top, h_idx.numpy(), h_val.numpy())

    def barrier():
        replicas.barrier(info)
        torch.cuda.synchronize()

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
    ms_e2e = replicas.max_over_ranks(ms_e2e, info, dev)
    same = bool(np.array_equal(h_ups.numpy(), d_ups.cpu().numpy()))
    census = tier_census(ctx, lambda: ctx.eval(d_params, N_seg, d_ups)) if rank == 0 else None
    issue = ctx.probe_fp32_issue(1 << 16) if rank == 0 else None
    wstruct = ctx.weight_structure()
    launches_total = int(leg["prof"]["kernel_launches"])
    ctx.destroy()

    # ---------------- second leg: the same bank with general per-pixel weights (12 B per pixel-eval) ----------------
    general = None
    if world == 1 and wstruct != 0 and not args.no_general_leg:
        ctx1 = api.Tfs(w.Nt, w.Nf, w.dt, weight_mode=1)
        ctx1.upload_data(coeff, weight, gap)
        leg1 = time_leg(api, torch, ctx1, w, d_params, n, N_seg, k_top, args.steps, warm, info, dev, True)
        general = (leg1, float(np.max(np.abs(leg1["d_ups"].cpu().numpy() - d_ups.cpu().numpy()) /
                                      np.maximum(d_ups.cpu().numpy(), 2.0 * N_seg))))
        ctx1.destroy()

    if rank != 0:
        replicas.finish(info)
        return 0

    secondary = {"error": sec_err} if sec_err else None
    if sec is not None:
        try:
            secondary = secondary_legs(api, torch, dev, sec, sec_ora)
        except Exception as exc:
            secondary = {"error": f"{type(exc).__name__}: {exc}"}
        secondary["oracle_seconds"] = sec_dt
        secondary["note"] = (f"each leg: 3 device-timed calls after 2 warm-up calls; parity = timed output vs oracle/ on the first "
                             f"{SEC_ROWS} rows of the leg's bank, criterion as in `parity`")

    peaks, peak_src = measured_peaks()
    sm_mhz = (clocks or {}).get("sm_mhz") or peaks.get("sm_max_mhz", 1965.0)
    terms, kern_ms, bytes_per_launch = roofline_terms(leg, args.steps, pixels, wstruct, l2_gbs, peaks, peak_src, sm_count, sm_mhz,
                                                      census, issue)
    # the larger of the byte term -- against the level that serves the gathers: shared memory for the slab
    # kernel -- and the arithmetic term (BASELINE.json north_star); the L1/L2 and HBM figures are context
    bound = "smem" if terms["smem"]["frac"] >= terms["alu"]["frac"] else "alu"
    prof = leg["prof"]
    n_launch = max(prof["eval_launches"], 1)
    line = {
        "metric": "templates/sec", "value": replicas.aggregate_rate(n, ms_step * 1e-3, info), "unit": "templates/s",
        "n_gpus": world, "steps": args.steps, "warmup": warm, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": cfg,
        "pixel_evals_per_sec": world * pixel_evals / (ms_step * 1e-3),
        "pixel_evals_per_template": pixel_evals / n,
        "active_pixel_histogram": pix_hist,
        "roofline": {"bound": bound, "kernel": "eval_list_kernel + eval_slab_kernel (one pair per step)",
                     "achieved": terms[bound]["achieved"],
                     "peak": terms[bound]["peak"], "peak_source": terms[bound]["peak_source"],
                     "unit": terms[bound]["unit"], "frac": terms[bound]["frac"], "traffic": None,
                     "algorithmic_bytes_per_launch": bytes_per_launch,
                     "algorithmic_bytes_per_pixel_eval": ALG_BYTES_PER_PIXEL_EVAL[wstruct],
                     "algorithmic_lane_ops_per_pixel": terms["alu"]["lane_ops_per_pixel"],
                     "weight_structure": wstruct, "kernel_ms_per_launch": kern_ms,
                     "slab_kernel_ms": prof["slab_kernel_ms"] / n_launch, "list_kernel_ms": prof["list_kernel_ms"] / n_launch,
                     "kernel_share_of_step": (prof["slab_kernel_ms"] + prof["list_kernel_ms"]) / leg["ms_total"],
                     "terms": terms},
        "cpu_baseline": cpu_baseline,
        "parity": parity,
        "secondary": secondary,
        "e2e": {"value": replicas.aggregate_rate(n, ms_e2e * 1e-3, info), "unit": "templates/s",
                "h2d_bytes_per_step": int(params.nbytes + h_ups.numpy().nbytes),
                "d2h_bytes_per_step": int(h_ups.numpy().nbytes + h_idx.numpy().nbytes + h_val.numpy().nbytes),
                "ms_per_step": ms_e2e, "matches_device_path": same},
        "gpu_launches": launches_total,
        "clocks": clocks,
    }
    if general is not None:
        leg1, dmax = general
        mhz1 = (leg1["clocks"] or {}).get("sm_mhz") or sm_mhz
        t1, k1, b1 = roofline_terms(leg1, args.steps, pixels, 0, l2_gbs, peaks, peak_src, sm_count, mhz1)
        line["general_weights_leg"] = {
            "what": "the same bank and data with tfs_opts.weight_mode = 1: W read next to every data pixel (12 B per pixel-eval)",
            "value": n / (leg1["ms_step"] * 1e-3), "unit": "templates/s", "ms_per_step": leg1["ms_step"],
            "kernel_ms_per_launch": k1, "algorithmic_bytes_per_launch": b1,
            "frac_smem": t1["smem"]["frac"], "frac_l2": t1["l2"]["frac"], "frac_alu": t1["alu"]["frac"],
            "max_norm_diff_vs_separable_leg": dmax, "clocks": leg1["clocks"]}
    extra = os.path.join(ROOT, "profiles", "roofline_traffic.json")      # ncu-derived, committed with the capture
    if os.path.exists(extra):
        try:
            t = json.load(open(extra)).get(w.name, {})
            # the capture is stamped with the hash of the kernel source it was taken at
            import hashlib
            src = os.path.join(ROOT, "paper_2510_19047_b200", "csrc", "tfs_kernels.cuh")
            cur = hashlib.sha256(open(src, "rb").read()).hexdigest()[:16]
            if t.get("kernel_source_sha256_16") == cur:
                line["roofline"].update({k: v for k, v in t.items() if k != "kernel_source_sha256_16"})
            else:
                line["roofline"].update({"traffic": None, "traffic_stale": True})
        except Exception:
            pass
    print(json.dumps(line))
    replicas.finish(info)
    return 0


if __name__ == "__main__":
    sys.exit(main())
