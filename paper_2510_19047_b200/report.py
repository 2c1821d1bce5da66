"""Throughput tables for the secondary BASELINE.json configurations (markdown on stdout).

    python -m paper_2510_19047_b200.report track-width     # configs[3]: throughput vs track width
    python -m paper_2510_19047_b200.report stress          # configs[3] at its stated size: 10^7 templates, batches of 2^20
    python -m paper_2510_19047_b200.report nseg            # configs[2]: N_seg swept over {1, 4, 16, 64}
    python -m paper_2510_19047_b200.report ladder          # configs[4]: the 64 -> 16 -> 4 -> 1 ladder at full size
    python -m paper_2510_19047_b200.report frontend        # NEXT-2: time series -> TF grid at the 2-year-shaped size
    python -m paper_2510_19047_b200.report window          # NEXT-2: window-aware template (tukey_alpha) vs the default
    python -m paper_2510_19047_b200.report search          # NEXT-4: tfs_eval_tseg and the per-tile lattice search
    python -m paper_2510_19047_b200.report channels        # NEXT-3: 1 / 2 / 3 channels, constant factors vs per-tranche transfer tables

Uses only the public binding (api.Tfs) and the seeded generators (synth); timing with CUDA events on
the current stream after warm-up, inputs resident on the device.  bench.py prints the headline line;
these tables are the "report throughput vs track width" / "N_seg swept" parts of the configs.
"""
from __future__ import annotations

import sys

import numpy as np


def _time_eval(ctx, torch, d_params, N_seg, reps=3, warm=2):
    n = d_params.shape[0]
    d_ups = torch.empty(n, dtype=torch.float32, device=d_params.device)
    for _ in range(warm):
        ctx.eval(d_params, N_seg, d_ups)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        ctx.eval(d_params, N_seg, d_ups)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def _counts(ctx, torch, d_params):
    c = torch.empty(d_params.shape[0], dtype=torch.int64, device=d_params.device)
    ctx.count_pixels(d_params, c)
    torch.cuda.synchronize()
    return c.cpu().numpy()


def _setup(name):
    import torch
    from . import api, synth
    assert torch.cuda.is_available(), "needs cuda:0 (libtfs has no CPU fallback)"
    torch.cuda.set_device(0)
    w = synth.WORKLOADS[name]
    coeff, weight, gap = synth.make_data(w)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    ctx.upload_data(coeff, weight, gap)
    return torch, api, synth, w, ctx, (coeff, weight, gap)


def track_width():
    torch, api, synth, w, ctx, data = _setup("cfg4")
    dev = torch.device("cuda:0")
    params = synth.make_templates(w)
    d_all = torch.from_numpy(params).to(dev)
    pix = _counts(ctx, torch, d_all)
    # active tranches per template from the window rule: pixels(H=10) - pixels(H=0) = 20 per active tranche
    ctx0 = api.Tfs(w.Nt, w.Nf, w.dt, half_width=0)
    ctx0.upload_data(*data)
    act = (pix - _counts(ctx0, torch, d_all)) // 20
    ctx0.destroy()
    width = np.where(act > 0, pix / np.maximum(act, 1), 0.0)
    print(f"# configs[3] (cfg4): throughput vs track width, N_seg = {w.N_seg}, grid {w.Nt} x {w.Nf}, "
          f"bank of {len(params)} (80 % as cfg2, 20 % merging inside the grid)\n")
    print("| sub-bank | templates | mean pixels / active tranche | mean active tranches | ms | templates/s | pixel-evals/s |")
    print("|---|---:|---:|---:|---:|---:|---:|")

    def row(label, p, px, ac):
        d = torch.from_numpy(np.ascontiguousarray(p)).to(dev)
        ms = _time_eval(ctx, torch, d, w.N_seg)
        print(f"| {label} | {len(p)} | {px.sum() / max(ac.sum(), 1):.1f} | {ac.mean():.0f} | {ms:.2f} | "
              f"{len(p) / ms * 1e3:.3e} | {2 * px.sum() / ms * 1e3:.3e} |")

    row("whole bank", params, pix, act)
    edges = [21, 21.5, 22, 23, 25, 30, 400]
    for a, b in zip(edges[:-1], edges[1:]):
        sel = (width >= a) & (width < b)
        if sel.sum() >= 1000:
            row(f"mean width in [{a}, {b})", params[sel], pix[sel], act[sel])
    # short tracks: the last days before a merger inside the grid, every tranche wide
    rng = np.random.default_rng(w.seed + 77)
    for days, mc_lo in ((30.0, 60.0), (10.0, 60.0), (4.0, 80.0), (2.0, 90.0)):
        p = synth.make_templates(w, n=200_000, seed=w.seed + int(days))
        p[:, 0] = np.exp(rng.uniform(np.log(mc_lo), np.log(100.0), len(p)))
        p[:, 1] = rng.uniform(0.3, 1.0, len(p)) * days * 86400.0
        d = torch.from_numpy(p).to(dev)
        px = _counts(ctx, torch, d)
        c0 = api.Tfs(w.Nt, w.Nf, w.dt, half_width=0)
        c0.upload_data(*data)
        ac = (px - _counts(c0, torch, d)) // 20
        c0.destroy()
        row(f"Mc in [{mc_lo:.0f}, 100], merger {0.3 * days:.1f}-{days:.0f} d after the data start", p, px, ac)
    ctx.destroy()


def stress():
    """configs[3] at its stated size: 10 batches of 2^20 templates (1.05 x 10^7) back to back, N_seg = 32, each batch its
    own seeded bank, resident on the device; sustained rate with the SM clock sampled during the run."""
    import subprocess
    import threading
    torch, api, synth, w, ctx, data = _setup("cfg4")
    dev = torch.device("cuda:0")
    banks = [torch.from_numpy(synth.make_templates(w, seed=w.seed + 100 * b)).to(dev) for b in range(10)]
    n = sum(b.shape[0] for b in banks)
    ups = torch.empty(banks[0].shape[0], dtype=torch.float32, device=dev)
    idx = torch.empty(banks[0].shape[0] // 100, dtype=torch.int64, device=dev)
    val = torch.empty(banks[0].shape[0] // 100, dtype=torch.float32, device=dev)
    for b in banks[:2]:
        ctx.eval(b, w.N_seg, ups)
    torch.cuda.synchronize()
    clocks = []
    proc = subprocess.Popen(["nvidia-smi", "-i", "0", "--query-gpu=clocks.sm,clocks_event_reasons.sw_power_cap,"
                             "clocks_event_reasons.hw_slowdown", "--format=csv,noheader,nounits", "-lms", "100"],
                            stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
    th = threading.Thread(target=lambda: clocks.extend(proc.stdout), daemon=True)
    th.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for rep in range(3):
        for b in banks:
            ctx.eval(b, w.N_seg, ups)
            ctx.topk(ups, idx.shape[0], idx, val)
    e1.record()
    torch.cuda.synchronize()
    proc.terminate()
    ms = e0.elapsed_time(e1) / 3
    mhz = [float(c.split(",")[0]) for c in clocks if c.strip()]
    flags = sorted({f.strip() for c in clocks for f in c.split(",")[1:] if "Active" in f and "Not" not in f})
    print(f"# configs[3] (cfg4) at its stated size: 10 batches of 2^20 = {n} templates, N_seg = {w.N_seg}, grid {w.Nt} x {w.Nf}\n")
    print(f"{ms:.1f} ms for the 10 batches (tfs_eval + tfs_topk of the top 1 % each; mean of 3 passes) = "
          f"{n / ms * 1e3:.3e} templates/s sustained; SM clock median {np.median(mhz) if mhz else float('nan'):.0f} MHz "
          f"over {len(mhz)} samples, throttle flags active: {flags or 'none'}")
    ctx.destroy()


def nseg():
    torch, api, synth, w, ctx, data = _setup("cfg3")
    dev = torch.device("cuda:0")
    n_valid = int(np.count_nonzero(data[2]))
    params = synth.make_templates(w)
    d = torch.from_numpy(params).to(dev)
    pix = _counts(ctx, torch, d)
    print(f"# configs[2] (cfg3): N_seg sweep, {len(params)} templates, grid {w.Nt} x {w.Nf}, "
          f"weight structure {ctx.weight_structure()}, {n_valid} valid tranches = {-(-n_valid // 64)} time tiles "
          f"of 64 for every N_seg\n")
    print("| N_seg | ms per tfs_eval | templates/s | pixel-evals/s |")
    print("|---:|---:|---:|---:|")
    for N in (1, 4, 16, 64):
        ms = _time_eval(ctx, torch, d, N)
        print(f"| {N} | {ms:.2f} | {len(params) / ms * 1e3:.3e} | {2 * pix.sum() / ms * 1e3:.3e} |")
    ctx.destroy()


def ladder_report():
    """Full-size configs[4]: 10^6 templates on the cfg5 grid, stages N_seg = 64, 16, 4, 1, top 1 % kept and
    replaced by 4 x 4 children per survivor.  Noise only (injections are made by the oracle, which this
    package never imports): this table times the stages; recovery is tested in tests/test_gpu_ladder.py."""
    torch, api, synth, w, ctx, _ = _setup("cfg5")
    from . import ladder
    dev = torch.device("cuda:0")
    d = torch.from_numpy(synth.make_templates(w)).to(dev)
    d_mc, d_tc = 2e-4, 1.0e4          # stage-0 lattice steps (relative Mc step, tc step in s)
    for _ in range(2):
        ladder.run(ctx, d, d_mc, d_tc)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    st = ladder.run(ctx, d, d_mc, d_tc)
    e1.record()
    torch.cuda.synchronize()
    print(f"# configs[4] (cfg5): ladder at full size, grid {w.Nt} x {w.Nf}, keep 1 %, 4 x 4 children per survivor\n")
    print(f"whole ladder (4 x tfs_eval + 4 x tfs_topk + 3 x tfs_refine): {e0.elapsed_time(e1):.2f} ms\n")
    print("| stage | N_seg | templates | kept | ms per tfs_eval | templates/s | best Upsilon |")
    print("|---:|---:|---:|---:|---:|---:|---:|")
    for i, s in enumerate(st):
        ms = _time_eval(ctx, torch, s.params, s.N_seg, reps=2, warm=1)
        print(f"| {i} | {s.N_seg} | {s.params.shape[0]} | {s.top_idx.shape[0]} | {ms:.2f} | "
              f"{s.params.shape[0] / ms * 1e3:.3e} | {float(s.top_val[0]):.1f} |")
    ctx.destroy()


def frontend_report():
    """tfs_upload_timeseries at the cfg3 size (2 channels x 4096 tranches x 6144 samples), device-resident input.
    The call = window + FFT + weights + gap mask (4 kernels) followed by the ordinary upload (pack, valid list,
    weight classification from the per-bin table) and a stream synchronisation.  Bytes that must cross HBM: read x and the
    mask, write and re-read D, write the packed grid (no per-pixel weight array exists on this path)."""
    import torch
    from . import api, synth
    torch.cuda.set_device(0)
    w = synth.WORKLOADS["cfg3"]
    x, mask, psd = synth.make_timeseries(w)
    dev = torch.device("cuda:0")
    tx, tm, tp = torch.from_numpy(x).to(dev), torch.from_numpy(mask).to(dev), torch.from_numpy(psd).to(dev)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    for _ in range(2):
        ctx.upload_timeseries(tx, tm, tp, 0.1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        ctx.upload_timeseries(tx, tm, tp, 0.1)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    npix = 2 * w.Nt * w.Nf
    mandatory = x.nbytes + mask.nbytes + 2 * npix * 8 + npix * 8        # read x and the mask; write and re-read D; write the grid
    print(f"# NEXT-2 front end at the cfg3 size: {w.Nt} tranches x {2 * w.Nf} samples x 2 channels\n")
    print(f"tfs_upload_timeseries (device input, Tukey 0.1, PSD weights, gap mask; includes the ordinary upload and "
          f"its synchronisation): {ms:.2f} ms per call; {mandatory / 1e9:.2f} GB must cross HBM "
          f"({mandatory / ms / 1e6:.0f} GB/s); weight structure {ctx.weight_structure()}, "
          f"{x.shape[1] * 2 / ms / 1e6:.1f} G samples/s")
    ctx.destroy()


def window_report():
    """The window-aware template (tfs_opts.tukey_alpha = 0.1) against the default on the same cfg3 data: every item
    goes through the list kernel and every pixel adds the two taper terms (twelve table look-ups)."""
    import torch
    from . import api, synth
    torch.cuda.set_device(0)
    dev = torch.device("cuda:0")
    w = synth.WORKLOADS["cfg3"]
    coeff, weight, gap = synth.make_data(w)
    d = torch.from_numpy(synth.make_templates(w, 200_000)).to(dev)
    print(f"# window-aware template on the cfg3 grid, {d.shape[0]} templates, N_seg = {w.N_seg}\n")
    print("| tukey_alpha | kernels | ms per tfs_eval | templates/s | pixel-evals/s |")
    print("|---|---|---:|---:|---:|")
    for alpha in (0.0, 0.1):
        ctx = api.Tfs(w.Nt, w.Nf, w.dt, tukey_alpha=alpha)
        ctx.upload_data(coeff, weight, gap)
        pix = _counts(ctx, torch, d)
        ms = _time_eval(ctx, torch, d, w.N_seg)
        print(f"| {alpha} | {'slab + list' if alpha == 0.0 else 'list, MODE 2'} | {ms:.2f} | {d.shape[0] / ms * 1e3:.3e} | "
              f"{2 * pix.sum() / ms * 1e3:.3e} |")
        ctx.destroy()


def search_report():
    """tfs_eval_tseg at the cfg3 size, and the tile search over a row of paper-sized tiles (5 Msun x 1e-4 Hz)
    on the cfg3 data (noise only): lattice 32 x 32 per tile, stages 16 -> 4 -> 1, 16 kept, 4 x 4 children, <= 3 extra levels."""
    import time
    torch, api, synth, w, ctx, _ = _setup("cfg3")
    from . import search
    dev = torch.device("cuda:0")
    d = torch.from_numpy(synth.make_templates(w)).to(dev)
    n = d.shape[0]
    ups = torch.empty(n, dtype=torch.float32, device=dev)
    neff = torch.empty(n, dtype=torch.int32, device=dev)
    print(f"# tfs_eval_tseg on the cfg3 grid ({w.Nt} tranches of {w.DT:.0f} s), {n} templates\n")
    print("| seg_tranches (T_seg) | N_seg | ms | templates/s | mean n_seg_eff |")
    print("|---:|---:|---:|---:|---:|")
    for M_tr in (256, 100, 30):
        for _ in range(2):
            ctx.eval_tseg(d, M_tr, ups, neff)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            ctx.eval_tseg(d, M_tr, ups, neff)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 3
        print(f"| {M_tr} ({M_tr * w.DT / 86400:.1f} d) | {-(-w.Nt // M_tr)} | {ms:.2f} | {n / ms * 1e3:.3e} | "
              f"{neff.float().mean().item():.2f} |")
    row = np.array([0.0, 0.0, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])
    tiles = [(25.0, 30.0, 8.0e-3 + 1e-4 * j, 8.1e-3 + 1e-4 * j) for j in range(16)]
    kw = dict(stages=(16, 4, 1), keep=16, r=4, max_extra=3, tol=1e-3)
    search.search_tiles(ctx, tiles[:2], row, 32, 32, **kw)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = search.search_tiles(ctx, tiles, row, 32, 32, **kw)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    nev = sum(l[1] for r_ in res for l in r_.levels)
    print(f"\n# tile search: {len(tiles)} tiles of 5 Msun x 1e-4 Hz at 8.0-9.6 mHz, noise only\n")
    print(f"{dt * 1e3:.1f} ms wall for {len(tiles)} tiles ({dt / len(tiles) * 1e3:.1f} ms per tile, {nev} template evaluations, "
          f"{sum(len(r_.levels) for r_ in res)} levels); hat-Upsilon_1 per tile: "
          + ", ".join(f"{r_.upsilon:.1f}" for r_ in res))
    ctx.destroy()


def channels_report():
    """Channels and transfer factors at the cfg3 size (Eq. 3 sums A, E, T; Eq. 29 T_alpha(f_nm) per tranche):
    the cfg3 bank on 1, 2 and 3 channels of cfg3-like noise, with the constant factors of `params` (tfs_eval) and with a
    16-knot complex table per template and channel interpolated at every tranche (tfs_eval_tf).  The third channel is a
    second pass over its own pair."""
    import torch
    from . import api, synth
    torch.cuda.set_device(0)
    dev = torch.device("cuda:0")
    w = synth.WORKLOADS["cfg3"]
    coeff, weight, gap = synth.make_data(w)
    n, K = 500_000, 16
    params = synth.make_templates(w, n)
    d = torch.from_numpy(params).to(dev)
    rng = np.random.default_rng(33)
    print(f"# channels and transfer factors on the cfg3 grid, {n} templates, N_seg = {w.N_seg}, {K} knots over 1-100 mHz\n")
    print("| channels | transfer factor | ms per call | templates/s | pixel-evals/s |")
    print("|---:|---|---:|---:|---:|")
    for C in (1, 2, 3):
        cc = np.ascontiguousarray(np.concatenate([coeff, coeff[:1]])[:C])
        ww = np.ascontiguousarray(np.concatenate([weight, weight[:1]])[:C])
        ctx = api.Tfs(w.Nt, w.Nf, w.dt, C)
        ctx.upload_data(cc, ww, gap)
        if C == 3:
            ctx.set_third_channel_factor(0.6, -0.3)          # constant T_T: the third channel is evaluated (a second pass)
        pix = _counts(ctx, torch, d)
        ups = torch.empty(n, dtype=torch.float32, device=dev)
        tab = torch.from_numpy(rng.standard_normal((n, C, K, 2)).astype(np.float32)).to(dev)
        for label, call in (("constant (params)", lambda: ctx.eval(d, w.N_seg, ups)),
                            ("table, interpolated per tranche", lambda: ctx.eval_tf(d, w.N_seg, tab, K, 1e-3, 6.6e-3, ups))):
            for _ in range(2):
                call()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(3):
                call()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 3
            print(f"| {C} | {label} | {ms:.2f} | {n / ms * 1e3:.3e} | {C * pix.sum() / ms * 1e3:.3e} |")
        ctx.destroy()


if __name__ == "__main__":
    what = sys.argv[1] if len(sys.argv) > 1 else ""
    if what == "track-width":
        track_width()
    elif what == "stress":
        stress()
    elif what == "nseg":
        nseg()
    elif what == "ladder":
        ladder_report()
    elif what == "frontend":
        frontend_report()
    elif what == "window":
        window_report()
    elif what == "search":
        search_report()
    elif what == "channels":
        channels_report()
    else:
        sys.exit(__doc__)
