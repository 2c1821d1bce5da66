"""Seeded synthetic inputs shaped like the paper's workloads.

Stand-ins for the Yorsh LDC data, which is not available: TF-domain noise,
per-pixel noise weights, gap masks and template-parameter banks for BASELINE.json configs 1-5.
This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, so it holds none
of the method's arithmetic: no track, no Fresnel kernel, no inner product.  Injected signals are
therefore NOT made here (tests add them with ``oracle.tfs_oracle.injection``); this module only
lists their parameters.  Generator: numpy ``default_rng(seed)`` (PCG64).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

YEAR_S = 365.25 * 86400.0
DAY_S = 86400.0


@dataclass(frozen=True)
class Workload:
    name: str
    Nt: int
    Nf: int
    dt: float
    n_templates: int
    N_seg: int
    seed: int
    noise: str                      # "white" | "psd" | "nonstat"
    gaps: bool
    mc_range: tuple = (5.0, 100.0)
    mc_dist: str = "log"            # "log" | "uniform"
    tc_range_yr: tuple = (0.0, 10.0)
    antenna: str = "sphere"         # "sphere" | "fixed"
    # (Mc, tc[yr], phic, (TA, TE) or None -> drawn, rho)
    injections: tuple = field(default_factory=tuple)

    @property
    def DT(self):
        return 2.0 * self.Nf * self.dt

    @property
    def df(self):
        return 1.0 / self.DT


WORKLOADS = {
    # BASELINE.json configs[0]
    "cfg1": Workload("cfg1", 512, 1024, 5.0, 64, 4, 0, "white", False, (25.0, 35.0), "uniform",
                     (0.3, 10.0), "fixed", ((30.0, 1.0, 0.3, (0.7 + 0j, 0.5 + 0j), 20.0),)),
    # configs[1]
    "cfg2": Workload("cfg2", 2048, 3072, 5.0, 100_000, 16, 1, "psd", False,
                     injections=((30.0, 6.0, 1.1, None, 12.0), (12.0, 3.0, 2.2, None, 15.0),
                                 (60.0, 2.5, 0.7, None, 25.0))),
    # configs[2]
    "cfg3": Workload("cfg3", 4096, 3072, 5.0, 1_000_000, 16, 2, "nonstat", True,
                     injections=((30.0, 6.0, 1.1, None, 12.0), (12.0, 4.5, 2.2, None, 15.0),
                                 (60.0, 5.0, 0.7, None, 25.0))),
    # configs[3]: one batch of 2^20; 80% as cfg2, 20% merging inside the grid (wide tracks)
    "cfg4": Workload("cfg4", 4096, 3072, 5.0, 1 << 20, 32, 3, "white", False),
    # configs[4]
    "cfg5": Workload("cfg5", 4096, 3072, 5.0, 1_000_000, 64, 4, "nonstat", True,
                     injections=((28.0, 7.0, 0.2, None, 14.0), (45.0, 5.5, 1.2, None, 13.0),
                                 (9.0, 6.5, 2.9, None, 13.5), (70.0, 4.8, 4.0, None, 12.0),
                                 (18.0, 9.0, 5.1, None, 11.0))),
}


def scaled(w: Workload, **kw) -> Workload:
    """Copy of a workload with some fields replaced (reduced sizes for parity tests)."""
    d = {k: getattr(w, k) for k in w.__dataclass_fields__}
    d.update(kw)
    return Workload(**d)


def sigma_model(w: Workload, rng):
    """Noise standard deviation per pixel, returned as (sig_t[Nt], sig_f[Nf]); sigma = outer."""
    sig_t = np.ones(w.Nt)
    sig_f = np.ones(w.Nf)
    if w.noise == "psd":
        # smooth PSD-like per-frequency weight: power law rising below 5 mHz
        f = np.arange(w.Nf) * w.df
        with np.errstate(divide="ignore"):
            sig_f = np.sqrt(1.0 + (5e-3 / f) ** 4)
        sig_f[0] = np.inf                                   # k = 0 carries zero weight
    elif w.noise == "nonstat":
        t = np.arange(w.Nt) * w.DT
        sig_t = 1.0 + 0.3 * np.sin(2.0 * np.pi * t / YEAR_S)
        glitch = rng.random(w.Nt) < 1e-3
        sig_t = np.where(glitch, 2.0 * sig_t, sig_t)
    return sig_t, sig_f


def gap_mask(w: Workload, rng):
    """uint8 [Nt], 1 = valid.  A 7 h gap every 14 days plus 20 random gaps of 1-10 days; a time
    bin is masked when it overlaps any gap."""
    g = np.ones(w.Nt, dtype=np.uint8)
    if not w.gaps:
        return g
    Tobs = w.Nt * w.DT
    starts = list(np.arange(14 * DAY_S, Tobs, 14 * DAY_S))
    lens = [7 * 3600.0] * len(starts)
    for _ in range(20):
        starts.append(rng.uniform(0.0, Tobs))
        lens.append(rng.uniform(1.0, 10.0) * DAY_S)
    for s, l in zip(starts, lens):
        m0 = int(np.floor(s / w.DT))
        m1 = int(np.ceil((s + l) / w.DT))
        g[max(m0, 0):min(m1, w.Nt)] = 0
    return g


def make_data(w: Workload, seed=None, dtype=np.float32):
    """Noise-only TF data.  Returns (coeff [2][Nt][Nf][2] re,im ; weight [2][Nt][Nf] ;
    gap [Nt] uint8).  re, im ~ N(0, sigma^2), weight = 1/sigma^2 (so E|D|^2 = 2/W)."""
    rng = np.random.default_rng(w.seed if seed is None else seed)
    sig_t, sig_f = sigma_model(w, rng)
    gap = gap_mask(w, rng)
    sig = (sig_t[:, None] * sig_f[None, :])
    finite = np.isfinite(sig)
    wt = np.where(finite, 1.0 / np.where(finite, sig, 1.0) ** 2, 0.0).astype(dtype)
    sig32 = np.where(finite, sig, 0.0).astype(dtype)
    coeff = np.empty((2, w.Nt, w.Nf, 2), dtype=dtype)
    for a in range(2):
        for m0 in range(0, w.Nt, 256):                      # chunked: bounded temporaries
            m1 = min(m0 + 256, w.Nt)
            z = rng.standard_normal((m1 - m0, w.Nf, 2), dtype=np.float32)
            coeff[a, m0:m1] = z * sig32[m0:m1, :, None]
    weight = np.broadcast_to(wt, (2, w.Nt, w.Nf)).copy()
    return coeff, weight, gap


def make_templates(w: Workload, n=None, seed=None):
    """Template bank [n][8] float64: Mc[Msun], tc[s], phic, TA.re, TA.im, TE.re, TE.im, amp."""
    n = w.n_templates if n is None else n
    rng = np.random.default_rng((w.seed if seed is None else seed) + 1000)
    p = np.empty((n, 8), dtype=np.float64)
    lo, hi = w.mc_range
    if w.mc_dist == "log":
        p[:, 0] = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    else:
        p[:, 0] = rng.uniform(lo, hi, n)
    p[:, 1] = rng.uniform(w.tc_range_yr[0], w.tc_range_yr[1], n) * YEAR_S
    p[:, 2] = rng.uniform(0.0, 2.0 * np.pi, n)
    if w.antenna == "fixed":
        p[:, 3:7] = (0.7, 0.0, 0.5, 0.0)
    else:
        v = rng.standard_normal((n, 4))                     # uniform on the sphere S^3
        p[:, 3:7] = v / np.linalg.norm(v, axis=1, keepdims=True)
    p[:, 7] = rng.uniform(0.5, 2.0, n)
    if w.name == "cfg4":
        # 20 %: heavy systems that merge inside the grid, so their last tranches sweep up to
        # hundreds of pixels (BASELINE.json configs[3]).  Interleaved so every batch has them.
        nw = n // 5
        idx = np.arange(nw) * 5
        p[idx, 0] = np.exp(rng.uniform(np.log(30.0), np.log(100.0), nw))
        p[idx, 1] = rng.uniform(0.0, 1.0, nw) * (w.Nt * w.DT)
    return p


def injection_params(w: Workload):
    """List of (params[8], rho) for the workload's injections (parameters only)."""
    rng = np.random.default_rng(w.seed + 2000)
    out = []
    for (mc, tc_yr, phic, T, rho) in w.injections:
        if T is None:
            v = rng.standard_normal(4)
            v /= np.linalg.norm(v)
        else:
            v = np.array([T[0].real, T[0].imag, T[1].real, T[1].imag])
        out.append((np.array([mc, tc_yr * YEAR_S, phic, v[0], v[1], v[2], v[3], 1.0]), rho))
    return out


def make_timeseries(w: Workload, seed=None):
    """Seeded real time series for the front end (tfs_upload_timeseries): x [2][Nt*2*Nf] float32 at cadence dt
    (white Gaussian noise of unit variance plus a few steady tones at frequencies that do not sit on a bin),
    a sample-validity mask [Nt*2*Nf] uint8 (6-hour gaps at random times adding up to 15 % of the samples, as
    in the paper's gap experiment P:297, plus a few short gaps inside tranches) and a smooth one-sided PSD model [2][Nf] (white level 2*dt with a red rise below
    5 mHz).  Inputs only: no window, no transform, no weights are formed here."""
    rng = np.random.default_rng((w.seed if seed is None else seed) + 3000)
    N = 2 * w.Nf
    ns = w.Nt * N
    x = rng.standard_normal((2, ns)).astype(np.float32)
    t = np.arange(ns, dtype=np.float64) * w.dt
    for a in range(2):
        for j in range(3):
            f = (0.13 + 0.27 * j + 0.05 * a) * 0.5 / w.dt * 0.9          # inside (0, Nyquist)
            x[a] += (3.0 / (1 + j) * np.cos(2 * np.pi * f * t + 0.3 * j + a)).astype(np.float32)
    mask = np.ones(ns, dtype=np.uint8)
    if w.gaps:
        # the paper's gap experiment: 6-hour gaps at random times, 15 % of the samples in total
        glen = max(1, int(round(6 * 3600.0 / w.dt)))
        for s in rng.integers(0, ns, size=max(1, int(round(0.15 * ns / glen)))):
            mask[s: s + glen] = 0
    for m in rng.choice(w.Nt, size=max(1, w.Nt // 16), replace=False):    # short gaps inside a tranche
        s = int(rng.integers(0, max(1, N - 8)))
        mask[m * N + s: min(m * N + s + int(rng.integers(1, 8)), (m + 1) * N)] = 0
    fk = np.arange(w.Nf) * w.df
    with np.errstate(divide="ignore"):
        S = 2.0 * w.dt * (1.0 + (5e-3 / fk) ** 4)
    S[0] = np.inf
    psd = np.stack([S, 1.7 * S]).astype(np.float32)
    return x, mask, psd
