"""CPU fp64 oracle for the time-frequency semi-coherent statistic Upsilon_Nseg.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import it.  It shares no code with the CUDA path (``paper_2510_19047_b200``)
and imports nothing from it.

It is a plain, slow, dense restatement of arXiv 2510.19047 ("Global time-frequency search for
stellar-mass binary black holes in LISA"), cited below as ``P:<line>`` = line of
``/root/reference/PAPER.md`` plus equation number, under the readings listed in ``DESIGN.md``
section 3 (``C1`` .. ``C16``).  Everything is numpy float64 / complex128.

What it computes, per template theta = (Mc, tc, phic, T_A, T_E, amp):
  1. the 0PN track at each tranche start t_m = m*DT                    (Eqs. 12-15)
  2. the Fresnel-kernel template pixels H[m, k] in the frequency window (Eqs. 16-22)
     materialised as a DENSE [Nt][Nf] complex128 array, zero outside the window
  3. z_n = sum_alpha T_alpha sum_{m in seg n} sum_{k=0}^{Nf-1} g[m] W conj(D) H   (Eq. 31, Eq. 30)
     hh_n = sum_alpha |T_alpha|^2 sum_m sum_k g[m] W |H|^2, summed over EVERY pixel
  4. P_n = |z_n|^2 / hh_n, Upsilon = sum_n P_n                          (Eq. 8, Eq. 9)

Pins (tests/test_oracle_pins.py, ``-m "not gpu"``): Fresnel values/derivative/quadrature (P1),
Eq. 16 against dt*FFT of a sampled linear chirp (P2), Parseval (P3), N_seg=1 == brute-force
phase-maximised coherent SNR^2 (P4), noiseless injection Upsilon_N = rho^2 (P5), time-domain
injection recovery (P6), noise-only E[Upsilon] = 2 N_eff (P7), Cauchy-Schwarz monotonicity
(P8), invariances (P9), gaps (P10), triple-loop re-implementation (P11), 21-bin power (P12).
Parity unpinned: nothing here reproduces the paper's search results (Figs. 4-6, Tables II-III);
the dataset, optimiser and LISA response are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

# GM_sun / c^3 in seconds (IAU nominal solar mass parameter / c^3).
MTSUN_S = 4.925490947e-6
YEAR_S = 365.25 * 86400.0


# ----------------------------------------------------------------------------------------------
# Fresnel integrals  C(z) = int_0^z cos(pi x^2/2) dx,  S(z) = int_0^z sin(pi x^2/2) dx
# ----------------------------------------------------------------------------------------------
_SERIES_MAX = 2.0      # |z| <= 2: Maclaurin series (largest term e^{2 pi} ~ 535 -> abs err ~1e-13)
_SERIES_TERMS = 40
_CF_DEPTH = 400        # Laplace continued fraction for erfc, evaluated bottom-up


def _fresnel_series(z):
    """Maclaurin series (Abramowitz & Stegun 7.3.11, 7.3.13; ref [52] of the paper)."""
    z = np.asarray(z, dtype=np.float64)
    a = 0.5 * math.pi * z * z          # pi z^2 / 2
    a2 = a * a
    # C = z * sum (-1)^n a^{2n} / ((2n)! (4n+1)) ;  S = z * sum (-1)^n a^{2n+1} / ((2n+1)! (4n+3))
    C = np.zeros_like(z)
    S = np.zeros_like(z)
    tc = np.ones_like(z)               # a^{2n}/(2n)!
    ts = a.copy()                      # a^{2n+1}/(2n+1)!
    sign = 1.0
    for n in range(_SERIES_TERMS):
        C += sign * tc / (4 * n + 1)
        S += sign * ts / (4 * n + 3)
        tc = tc * a2 / ((2 * n + 1) * (2 * n + 2))
        ts = ts * a2 / ((2 * n + 2) * (2 * n + 3))
        sign = -sign
    return z * C, z * S


def _fresnel_cf(z):
    """z > 0.  C + iS = (1+i)/2 * erf(w), w = sqrt(pi)/2 (1-i) z  (A&S 7.3.22), with
    erfc(w) = exp(-w^2)/sqrt(pi) * 1/(w + (1/2)/(w + 1/(w + (3/2)/(w + ...))))  (A&S 7.1.14),
    the continued fraction evaluated bottom-up to fixed depth.  exp(-w^2) = exp(i pi z^2/2)."""
    z = np.asarray(z, dtype=np.float64)
    w = (0.5 * math.sqrt(math.pi)) * (1.0 - 1.0j) * z
    t = w.copy()
    for k in range(_CF_DEPTH, 0, -1):
        t = w + (0.5 * k) / t
    ph = 0.5 * math.pi * np.mod(z * z, 4.0)          # exp(i pi z^2/2) has period 4 in z^2
    erfc = (np.cos(ph) + 1j * np.sin(ph)) / (math.sqrt(math.pi) * t)
    cs = 0.5 * (1.0 + 1.0j) * (1.0 - erfc)
    return cs.real, cs.imag


def fresnel_cs(z):
    """Exact (to ~1e-13) Fresnel integrals C(z), S(z) for real z of any sign; odd in z."""
    z = np.asarray(z, dtype=np.float64)
    az = np.abs(z)
    C = np.empty_like(az)
    S = np.empty_like(az)
    small = az <= _SERIES_MAX
    if np.any(small):
        C[small], S[small] = _fresnel_series(az[small])
    big = ~small
    if np.any(big):
        fin = big & np.isfinite(az)
        if np.any(fin):
            C[fin], S[fin] = _fresnel_cf(az[fin])
        inf = big & ~np.isfinite(az)
        C[inf] = 0.5
        S[inf] = 0.5
    sg = np.sign(z)
    return sg * C, sg * S


def fresnel_cs_paper(z):
    """The paper's own approximants, verbatim: Eqs. 23-24 for |z| > 6, Eqs. 25-28 for |z| <= 6
    (P:184-207), odd-extended.  NOT accurate to the claimed 1e-4 (C8)."""
    z = np.asarray(z, dtype=np.float64)
    a = np.abs(z)
    ph = 0.5 * math.pi * np.mod(a * a, 4.0)
    cz, sz = np.cos(ph), np.sin(ph)
    with np.errstate(divide="ignore", invalid="ignore"):
        S_big = 0.5 - cz / (math.pi * a)                                   # Eq. 23
        C_big = 0.5 + sz / (math.pi * a)                                   # Eq. 24
    f = (1.0 + 0.926 * a) / (2.0 + 1.792 * a + 3.104 * a * a)              # Eq. 27
    g = 1.0 / (2.0 + 4.142 * a + 3.492 * a * a + 6.670 * a ** 3)           # Eq. 28
    S_small = 0.5 - f * cz - g * sz                                        # Eq. 25
    C_small = 0.5 + f * sz - g * cz                                        # Eq. 26
    big = a > 6.0
    C = np.where(big, C_big, C_small)
    S = np.where(big, S_big, S_small)
    sg = np.sign(z)
    return sg * C, sg * S


# ----------------------------------------------------------------------------------------------
# Grid, options, template parameters
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Grid:
    """TF grid geometry (C1): Nt tranches of length DT = 2*Nf*dt, Nf bins of width
    df = 1/DT; tranche m starts at t_m = m*DT; bin k sits at f_k = k*df."""
    Nt: int
    Nf: int
    dt: float

    @property
    def DT(self) -> float:
        return 2.0 * self.Nf * self.dt

    @property
    def df(self) -> float:
        return 1.0 / self.DT

    @property
    def Tobs(self) -> float:
        return self.Nt * self.DT


@dataclass(frozen=True)
class Opts:
    """Mirror of ``tfs_opts`` in include/tfs.h.  f_lo/f_hi None -> [1*df, (Nf-1)*df]."""
    half_width: int = 10          # H; N_F = 2H+1 = 21
    adaptive_width: int = 1       # k_hi = ceil(x+c)+H (C4); 0 = paper-strict ceil(x)+H
    c_max: float = 300.0          # tranches with fdot*DT^2 > c_max are skipped
    f_lo: float | None = None
    f_hi: float | None = None
    fresnel_mode: int = 0         # 0 exact C,S ; 1 the paper's Eqs. 23-28 verbatim
    tukey_alpha: float = 0.0      # > 0: window-aware template for Tukey(alpha)-windowed tranches (C2/C24)

    def band(self, grid: Grid):
        lo = grid.df if self.f_lo is None else self.f_lo
        hi = (grid.Nf - 1) * grid.df if self.f_hi is None else self.f_hi
        return lo, hi


def segment_of_bin(m, Nt: int, N_seg: int):
    """n(m) = floor(m * N_seg / Nt): N_seg equal-index segments over [0, T_obs) (C9)."""
    return (np.asarray(m, dtype=np.int64) * N_seg) // Nt


def segment_of_bin_tseg(m, seg_tranches: int):
    """n(m) = floor(m / M_tr): segments of fixed duration T_seg = M_tr DT laid from the start of the data,
    t_n = n T_seg (M_tr = T_seg/DT tranches per segment).  N_seg = ceil(Nt / M_tr)."""
    return np.asarray(m, dtype=np.int64) // int(seg_tranches)


# ----------------------------------------------------------------------------------------------
# Step 1-2: 0PN track and window per tranche
# ----------------------------------------------------------------------------------------------
def track(Mc_msun: float, tc: float, phic: float, amp: float, grid: Grid, opts: Opts, gap_mask=None):
    """Track quantities at every tranche start (Eqs. 12-15, evaluated at t_nm, C6).

    0PN chirp (textbook closed form, C5), M = Mc*GMsun/c^3, tau = tc - t_m,
    X = tau/(5M):  f = X^{-3/8}/(8 pi M);  phi = phic - 2 X^{5/8};  fdot = 3 f/(8 tau);
    A = amp * f^{2/3}.  Returns a dict of length-Nt arrays; inactive tranches have active=False.
    """
    m = np.arange(grid.Nt, dtype=np.float64)
    DT, df = grid.DT, grid.df
    M = Mc_msun * MTSUN_S
    tau = tc - m * DT
    ok = tau > DT                                       # whole tranche precedes coalescence
    if gap_mask is not None:
        ok = ok & (np.asarray(gap_mask) != 0)           # C10: tranches overlapping a gap dropped
    ok = ok & np.isfinite(tau)
    tau_s = np.where(ok, tau, 1.0)
    X = tau_s / (5.0 * M)
    f = X ** (-0.375) / (8.0 * math.pi * M)
    phi = phic - 2.0 * X ** 0.625
    fdot = 3.0 * f / (8.0 * tau_s)
    A = amp * f ** (2.0 / 3.0)
    x = f * DT                                          # track position in bins
    c = fdot * DT * DT                                  # bins swept in one tranche
    f_lo, f_hi = opts.band(grid)
    active = ok & (f >= f_lo) & (f + fdot * DT <= f_hi) & (c <= opts.c_max)
    H = opts.half_width
    kc = np.ceil(x)                                     # "nearest frequency bin above f_nm" (C3)
    k_lo = kc - H
    k_hi = (np.ceil(x + c) if opts.adaptive_width else kc) + H
    k_lo = np.clip(k_lo, 1, grid.Nf - 1).astype(np.int64)
    k_hi = np.clip(k_hi, 1, grid.Nf - 1).astype(np.int64)
    return dict(active=active, f=f, fdot=fdot, phi=phi, A=A, x=x, c=c, k_lo=k_lo, k_hi=k_hi)


# ----------------------------------------------------------------------------------------------
# Step 3: Fresnel-kernel template pixels (Eq. 16)
# ----------------------------------------------------------------------------------------------
def kernel_pixels(x, c, phi, A, k, fresnel_mode: int = 0):
    """h~_nm(f_k)/DT at bins k (Eqs. 16-22); x, c, phi, A scalars or arrays shaped like k.

    With u = x - k = (f_nm - f_k)/df:  zeta = u df / fdot (Eq. 17),  pi fdot zeta^2 = pi u^2 / c,
    v(t_nm) = sqrt(2 fdot) zeta = sqrt(2/c) u,  v(t_nm+1) = sqrt(2/c) (u + c) (Eq. 22), and
    1/sqrt(2 fdot) = DT / sqrt(2c).  The common factor DT is dropped on both sides (C16).
    """
    k = np.asarray(k, dtype=np.float64)
    u = x - k
    s = np.sqrt(2.0 / c)
    v0 = s * u
    v1 = s * (u + c)
    fr = fresnel_cs_paper if fresnel_mode == 1 else fresnel_cs
    C1, S1 = fr(v1)
    C0, S0 = fr(v0)
    F = (C1 - C0) + 1j * (S1 - S0)                                          # Eqs. 19-21
    ph = phi - math.pi * u * u / c
    return (A / np.sqrt(2.0 * c)) * (np.cos(ph) + 1j * np.sin(ph)) * F     # Eq. 16


# ----------------------------------------------------------------------------------------------
# Window-aware template pixels: the tranche is Tukey-windowed before its Fourier transform
# ----------------------------------------------------------------------------------------------
def tukey_profile(s, alpha: float):
    """Tukey (tapered-cosine) window as a function of the position s in [0, 1] inside the tranche, shape
    parameter alpha = fraction of the tranche inside the two cosine tapers ("Tukey-windowed with a shape
    parameter of 0.1"; reading C24: the continuous profile, the O(1/N) difference to a sampled window is dropped)."""
    s = np.asarray(s, dtype=np.float64)
    if alpha <= 0.0:
        return np.ones_like(s)
    ell = 0.5 * min(alpha, 1.0)
    w = np.ones_like(s)
    lo = s < ell
    hi = s > 1.0 - ell
    w[lo] = 0.5 * (1.0 - np.cos(math.pi * s[lo] / ell))
    w[hi] = 0.5 * (1.0 - np.cos(math.pi * (1.0 - s[hi]) / ell))
    return w


_GL_NODES, _GL_WEIGHTS = np.polynomial.legendre.leggauss(16)


def kernel_pixels_windowed_quad(x, c, phi, A, k, alpha: float):
    """THE DEFINITION: h~_nm(f_k)/DT for a tranche multiplied by the Tukey(alpha) window before its Fourier
    transform, by direct quadrature of

        A exp(i phi) int_0^1 w(s) exp{i (2 pi u s + pi c s^2)} ds,    u = x - k,

    i.e. Eq. 16's integrand (phase Taylor-expanded about the tranche start, Eqs. 12-15, in units s = t/DT)
    times w(s).  Composite 16-point Gauss-Legendre on [0, l], [l, 1-l], [1-l, 1] (l = alpha/2), panels short enough
    that the phase advances by less than ~2 rad per panel.  Slow: for pins and small cases."""
    x, c, phi, A, k = np.broadcast_arrays(*(np.asarray(v, dtype=np.float64) for v in (x, c, phi, A, k)))
    shape = k.shape
    u = (x - k).ravel()[:, None]
    cc = c.ravel()[:, None]
    ell = 0.5 * min(max(alpha, 0.0), 1.0)
    cuts = [0.0, 1.0] if ell == 0.0 else sorted({0.0, ell, 1.0 - ell, 1.0})
    total = np.zeros(u.shape[0], dtype=np.complex128)
    rate = float(np.max(2.0 * math.pi * (np.abs(u) + cc)))             # max |d phase / ds| of the chirp
    for s0, s1 in zip(cuts[:-1], cuts[1:]):
        taper = ell > 0.0 and (s1 <= ell or s0 >= 1.0 - ell)           # the cosine adds pi of argument over a taper
        npan = 1 + int(math.ceil((rate * (s1 - s0) + (math.pi if taper else 0.0)) / 2.0))
        edges = np.linspace(s0, s1, npan + 1)
        h = 0.5 * (edges[1:] - edges[:-1])[:, None]
        mid = 0.5 * (edges[1:] + edges[:-1])[:, None]
        s = (mid + h * _GL_NODES[None, :]).ravel()[None, :]                 # [1][nodes]
        wq = (h * _GL_WEIGHTS[None, :]).ravel()[None, :]
        for i0 in range(0, u.shape[0], 64):                                 # pixels in blocks (memory)
            ub, cb = u[i0:i0 + 64], cc[i0:i0 + 64]
            f = tukey_profile(s, alpha) * np.exp(1j * (2.0 * math.pi * ub * s + math.pi * cb * s * s))
            total[i0:i0 + 64] += np.sum(wq * f, axis=1)
    out = A.ravel() * (np.cos(phi.ravel()) + 1j * np.sin(phi.ravel())) * total
    return out.reshape(shape)


def _chirp_integral(u, c, s0: float, s1: float):
    """I(u; s0, s1) = int_{s0}^{s1} exp{i (2 pi u s + pi c s^2)} ds in Fresnel integrals: completing the square,
    2 pi u s + pi c s^2 = pi v^2/2 - pi u^2/c with v = sqrt(2/c) (u + c s) (Eq. 22 at a general time), so
    I = exp(-i pi u^2/c) [F(v(s1)) - F(v(s0))] / sqrt(2c),  F = C + iS  (Eqs. 16-21 with other end points)."""
    sq = np.sqrt(2.0 / c)
    C1, S1 = fresnel_cs(sq * (u + c * s1))
    C0, S0 = fresnel_cs(sq * (u + c * s0))
    ph = -math.pi * np.mod(u * u / c, 2.0)
    return (np.cos(ph) + 1j * np.sin(ph)) * ((C1 - C0) + 1j * (S1 - S0)) / np.sqrt(2.0 * c)


def kernel_pixels_windowed(x, c, phi, A, k, alpha: float):
    """The same quantity in closed form (pinned against kernel_pixels_windowed_quad).  With l = alpha/2, b = 1/alpha,
    the window is 1 minus the two taper deficits [1 + cos(2 pi b s)]/2 on [0, l] and [1 + cos(2 pi b (1-s))]/2 on
    [1-l, 1]; a cosine shifts u by +-b, so

        K_w(u) = I(u;0,1) - [ I(u;0,l)/2 + I(u+b;0,l)/4 + I(u-b;0,l)/4 ]
                          - [ I(u;1-l,1)/2 + e^{-2 pi i b} I(u+b;1-l,1)/4 + e^{+2 pi i b} I(u-b;1-l,1)/4 ]."""
    k = np.asarray(k, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    u = x - k
    K = _chirp_integral(u, c, 0.0, 1.0)
    if alpha > 0.0:
        a = min(alpha, 1.0)
        ell, b = 0.5 * a, 1.0 / a
        eb = complex(math.cos(2.0 * math.pi * b), math.sin(2.0 * math.pi * b))
        K = K - (0.5 * _chirp_integral(u, c, 0.0, ell) + 0.25 * _chirp_integral(u + b, c, 0.0, ell)
                 + 0.25 * _chirp_integral(u - b, c, 0.0, ell))
        K = K - (0.5 * _chirp_integral(u, c, 1.0 - ell, 1.0) + 0.25 * np.conj(eb) * _chirp_integral(u + b, c, 1.0 - ell, 1.0)
                 + 0.25 * eb * _chirp_integral(u - b, c, 1.0 - ell, 1.0))
    return np.asarray(A) * (np.cos(phi) + 1j * np.sin(phi)) * K


def dense_template(Mc_msun, tc, phic, amp, grid: Grid, opts: Opts, gap_mask=None, truncate=True):
    """Dense [Nt][Nf] complex128 template (without T_alpha), zero outside each tranche's window.

    truncate=False fills every bin 1..Nf-1 of each active tranche (used for injections and for
    the Parseval pin); truncate=True is the method's window (C3/C4).
    """
    tr = track(Mc_msun, tc, phic, amp, grid, opts, gap_mask)
    Hd = np.zeros((grid.Nt, grid.Nf), dtype=np.complex128)
    ms = np.nonzero(tr["active"])[0]
    if ms.size == 0:
        return Hd
    lo = tr["k_lo"][ms] if truncate else np.full(ms.size, 1)
    hi = tr["k_hi"][ms] if truncate else np.full(ms.size, grid.Nf - 1)
    # all window pixels of all active tranches, flattened: (mm[i], kk[i])
    mm = np.repeat(ms, hi - lo + 1)
    kk = np.concatenate([np.arange(l, h + 1) for l, h in zip(lo, hi)])
    if opts.tukey_alpha > 0.0:
        Hd[mm, kk] = kernel_pixels_windowed(tr["x"][mm], tr["c"][mm], tr["phi"][mm], tr["A"][mm], kk,
                                            opts.tukey_alpha)
    else:
        Hd[mm, kk] = kernel_pixels(tr["x"][mm], tr["c"][mm], tr["phi"][mm], tr["A"][mm], kk,
                                   opts.fresnel_mode)
    return Hd


def window_pixel_counts(Mc_msun, tc, grid: Grid, opts: Opts, gap_mask=None):
    """Number of window pixels (k_hi-k_lo+1 summed over active tranches) of one template."""
    tr = track(Mc_msun, tc, 0.0, 1.0, grid, opts, gap_mask)
    a = tr["active"]
    return int(np.sum((tr["k_hi"] - tr["k_lo"] + 1)[a]))


# ----------------------------------------------------------------------------------------------
# Steps 4-5: dense inner products, segment combine
# ----------------------------------------------------------------------------------------------
def segment_products(Hd, T, D, W, gap_mask, N_seg: int, seg=None):
    """z_n and hh_n by dense sums over EVERY pixel of every channel (Eq. 31, Eq. 30).

    Hd [Nt][Nf] complex128; T [C] complex (transfer factors, Eq. 29, constant per
    template under C5/A12) or [C][Nt] complex (one factor per tranche: T_alpha(f_nm), "computed
    once per tranche for all frequency bins"); D [C][Nt][Nf] complex; W [C][Nt][Nf] real >= 0
    (or None => 1); gap_mask [Nt] (or None).  W stands for 4 df / S so that
    Upsilon = |sum W conj(D) y|^2 / sum W |y|^2.  seg [Nt] = segment of each tranche (default: segment_of_bin).
    """
    Cn, Nt, Nf = D.shape
    g = np.ones(Nt) if gap_mask is None else (np.asarray(gap_mask) != 0).astype(np.float64)
    if seg is None:
        seg = segment_of_bin(np.arange(Nt), Nt, N_seg)
    z = np.zeros(N_seg, dtype=np.complex128)
    hh = np.zeros(N_seg, dtype=np.float64)
    H2 = (Hd.real ** 2 + Hd.imag ** 2)
    for a in range(Cn):
        Da = D[a].astype(np.complex128)
        Wa = np.ones((Nt, Nf)) if W is None else W[a].astype(np.float64)
        zm = np.sum(Wa * np.conj(Da) * Hd, axis=1) * g          # per-tranche (d_nm | h_nm)
        qm = np.sum(Wa * H2, axis=1) * g
        if np.ndim(T[a]) == 0:
            z += T[a] * np.bincount(seg, weights=zm.real, minlength=N_seg)
            z += T[a] * 1j * np.bincount(seg, weights=zm.imag, minlength=N_seg)
            hh += abs(T[a]) ** 2 * np.bincount(seg, weights=qm, minlength=N_seg)
        else:
            Ta = np.asarray(T[a], dtype=np.complex128)           # [Nt]: the factor of each tranche
            tz = Ta * zm
            z += np.bincount(seg, weights=tz.real, minlength=N_seg)
            z += 1j * np.bincount(seg, weights=tz.imag, minlength=N_seg)
            hh += np.bincount(seg, weights=np.abs(Ta) ** 2 * qm, minlength=N_seg)
    return z, hh


def combine(z, hh):
    """P_n = |z_n|^2/hh_n (0 where hh_n = 0); Upsilon = sum_n P_n (Eq. 8, Eq. 9)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        P = np.where(hh > 0, (z.real ** 2 + z.imag ** 2) / hh, 0.0)
    return P, float(np.sum(P))


PARAM_COLS = 8    # Mc[Msun], tc[s], phic, TA.re, TA.im, TE.re, TE.im, amp   (include/tfs.h)


def evaluate(params, D, W, gap_mask, grid: Grid, N_seg: int, opts: Opts = Opts()):
    """Upsilon for every row of params [n][8].  Returns dict(upsilon[n], seg_power[n][N_seg],
    seg_dh[n][N_seg] complex, seg_hh[n][N_seg]).  Rows with NaN/Inf give all zeros."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    n = params.shape[0]
    ups = np.zeros(n)
    segP = np.zeros((n, N_seg))
    segz = np.zeros((n, N_seg), dtype=np.complex128)
    segh = np.zeros((n, N_seg))
    for i in range(n):
        p = params[i]
        if not np.all(np.isfinite(p)) or p[0] <= 0:
            continue
        Hd = dense_template(p[0], p[1], p[2], p[7], grid, opts, gap_mask, truncate=True)
        T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6], 0.0])   # a third channel has no column: T_T = 0
        z, hh = segment_products(Hd, T[: D.shape[0]], D, W, gap_mask, N_seg)
        P, U = combine(z, hh)
        ups[i], segP[i], segz[i], segh[i] = U, P, z, hh
    return dict(upsilon=ups, seg_power=segP, seg_dh=segz, seg_hh=segh)


def evaluate_tseg(params, D, W, gap_mask, grid: Grid, seg_tranches: int, opts: Opts = Opts()):
    """As evaluate, with segments of fixed duration T_seg = seg_tranches * DT (segment_of_bin_tseg);
    N_seg = ceil(Nt / seg_tranches).  Also returns n_seg_eff[n] = number of segments with hh_n > 0: the paper's
    template-dependent N_seg = tau / T_seg, tau = min(T_obs, t_c), counted on the grid."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    n = params.shape[0]
    N_seg = -(-grid.Nt // int(seg_tranches))
    seg = segment_of_bin_tseg(np.arange(grid.Nt), seg_tranches)
    ups = np.zeros(n)
    neff = np.zeros(n, dtype=np.int64)
    segP = np.zeros((n, N_seg))
    segz = np.zeros((n, N_seg), dtype=np.complex128)
    segh = np.zeros((n, N_seg))
    for i in range(n):
        p = params[i]
        if not np.all(np.isfinite(p)) or p[0] <= 0:
            continue
        Hd = dense_template(p[0], p[1], p[2], p[7], grid, opts, gap_mask, truncate=True)
        T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6], 0.0])
        z, hh = segment_products(Hd, T[: D.shape[0]], D, W, gap_mask, N_seg, seg=seg)
        P, U = combine(z, hh)
        ups[i], segP[i], segz[i], segh[i], neff[i] = U, P, z, hh, int(np.sum(hh > 0))
    return dict(upsilon=ups, n_seg_eff=neff, seg_power=segP, seg_dh=segz, seg_hh=segh)


# ----------------------------------------------------------------------------------------------
# Frequency-dependent transfer factor per tranche (Eq. 7, Eq. 29)
# ----------------------------------------------------------------------------------------------
def transfer_at(table, f_knot0: float, f_knot_step: float, f):
    """T(f) from a table of K complex values at the knots f_knot0 + j f_knot_step: linear between knots,
    held at the end values outside them (include/tfs.h, tfs_eval_tf); K = 1 is a constant."""
    table = np.asarray(table, dtype=np.complex128)
    f = np.asarray(f, dtype=np.float64)
    K = table.shape[-1]
    if K == 1:
        return np.broadcast_to(table[..., 0], f.shape).astype(np.complex128)
    s = np.clip((f - f_knot0) / f_knot_step, 0.0, K - 1.0)
    j = np.minimum(np.floor(s).astype(np.int64), K - 2)
    t = s - j
    return table[..., j] * (1.0 - t) + table[..., j + 1] * t


def evaluate_tf(params, tables, f_knot0, f_knot_step, D, W, gap_mask, grid: Grid, N_seg: int, opts: Opts = Opts()):
    """As evaluate, with the transfer factor of channel alpha in tranche m read from the template's table
    at the tranche-start frequency f_m (C6): T_alpha,m = transfer_at(tables[i, alpha], ..., f_m).
    tables [n][C][K] complex.  The T columns of params are ignored."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    tables = np.asarray(tables, dtype=np.complex128)
    n = params.shape[0]
    Cn = D.shape[0]
    ups = np.zeros(n)
    segP = np.zeros((n, N_seg))
    segz = np.zeros((n, N_seg), dtype=np.complex128)
    segh = np.zeros((n, N_seg))
    for i in range(n):
        p = params[i]
        if not np.all(np.isfinite(p)) or p[0] <= 0:
            continue
        Hd = dense_template(p[0], p[1], p[2], p[7], grid, opts, gap_mask, truncate=True)
        tr = track(p[0], p[1], p[2], p[7], grid, opts, gap_mask)
        T = [transfer_at(tables[i, a], f_knot0, f_knot_step, tr["f"]) for a in range(Cn)]
        z, hh = segment_products(Hd, T, D, W, gap_mask, N_seg)
        P, U = combine(z, hh)
        ups[i], segP[i], segz[i], segh[i] = U, P, z, hh
    return dict(upsilon=ups, seg_power=segP, seg_dh=segz, seg_hh=segh)


def injection_tf(p, table, f_knot0, f_knot_step, rho: float, W, gap_mask, grid: Grid, opts: Opts = Opts(),
                 truncate=False):
    """As injection, for a source whose channel alpha carries T_alpha(f_m) from `table` [C][K] in tranche m."""
    Hd = dense_template(p[0], p[1], p[2], p[7], grid, opts, None, truncate=truncate)
    tr = track(p[0], p[1], p[2], p[7], grid, opts, None)
    table = np.asarray(table, dtype=np.complex128)
    S = np.stack([transfer_at(table[a], f_knot0, f_knot_step, tr["f"])[:, None] * Hd for a in range(table.shape[0])])
    g = np.ones(grid.Nt) if gap_mask is None else (np.asarray(gap_mask) != 0).astype(np.float64)
    Wd = np.ones_like(S.real) if W is None else W.astype(np.float64)
    norm2 = float(np.sum(Wd * (S.real ** 2 + S.imag ** 2) * g[None, :, None]))
    S *= rho / math.sqrt(norm2)
    return S * g[None, :, None]


def topk(upsilon, k: int):
    """Indices and values of the k largest; stable descending (ties -> lower index)."""
    u = np.asarray(upsilon)
    idx = np.argsort(-u, kind="stable")[:k]
    return idx.astype(np.int64), u[idx]


# ----------------------------------------------------------------------------------------------
# Injection (data generation for tests; uses the dense UNtruncated template)
# ----------------------------------------------------------------------------------------------
def injection(p, rho: float, W, gap_mask, grid: Grid, opts: Opts = Opts(), truncate=False):
    """Dense template (untruncated by default) of parameters p[8], per channel, scaled so that
    sum_alpha |T_alpha|^2 sum W |H|^2 = rho^2 over non-gap tranches.  Returns S [C][Nt][Nf]
    complex128 to be ADDED to the data (signal present inside gaps is removed with the data)."""
    Hd = dense_template(p[0], p[1], p[2], p[7], grid, opts, None, truncate=truncate)
    T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6], 0.0])          # a third channel has no column: T_T = 0
    Cn = 2 if W is None else W.shape[0]
    S = np.stack([T[a] * Hd for a in range(Cn)])
    g = np.ones(grid.Nt) if gap_mask is None else (np.asarray(gap_mask) != 0).astype(np.float64)
    Wd = np.ones_like(S.real) if W is None else W.astype(np.float64)
    norm2 = float(np.sum(Wd * (S.real ** 2 + S.imag ** 2) * g[None, :, None]))
    S *= rho / math.sqrt(norm2)
    return S * g[None, :, None]


# ----------------------------------------------------------------------------------------------
# N_seg ladder (BASELINE.json configs[4]; hierarchical N_seg reduction; C19)
# ----------------------------------------------------------------------------------------------
def refine(params, idx, r: int, d_mc_rel: float, d_tc: float):
    """r*r children per survivor on a lattice r times denser per dimension that tiles the parent's
    (Mc, tc) cell of size (Mc d_mc_rel) x d_tc:  o_i = (2i+1-r)/(2r);  child (a, b) of parent j at
    row j r^2 + a r + b:  Mc' = Mc (1 + o_a d_mc_rel),  tc' = tc + o_b d_tc,  rest copied."""
    params = np.asarray(params, dtype=np.float64)
    out = np.empty((len(idx) * r * r, PARAM_COLS), dtype=np.float64)
    row = 0
    for j in idx:
        p = params[int(j)]
        for a in range(r):
            oa = np.float64(2 * a + 1 - r) / np.float64(2 * r)
            for b in range(r):
                ob = np.float64(2 * b + 1 - r) / np.float64(2 * r)
                out[row] = p
                out[row, 0] = p[0] * (1.0 + oa * d_mc_rel)
                out[row, 1] = p[1] + ob * d_tc
                row += 1
    return out


def ladder(params, D, W, gap_mask, grid: Grid, d_mc_rel: float, d_tc: float, stages=(64, 16, 4, 1),
           keep_frac: float = 0.01, r: int = 4, keep_min: int = 1, opts: Opts = Opts()):
    """Stage s: evaluate at N_seg = stages[s], keep the top ceil(keep_frac n) (at least keep_min),
    refine each survivor r x r with the steps divided by r per stage.  Returns a list of dicts
    (N_seg, params, upsilon, top_idx, top_val, d_mc_rel, d_tc), one per stage."""
    out = []
    cur = np.asarray(params, dtype=np.float64)
    for s, N_seg in enumerate(stages):
        ups = evaluate(cur, D, W, gap_mask, grid, N_seg, opts)["upsilon"]
        n = len(cur)
        k = min(n, max(keep_min, int(math.ceil(keep_frac * n))))
        idx, val = topk(ups, k)
        out.append(dict(N_seg=N_seg, params=cur, upsilon=ups, top_idx=idx, top_val=val,
                        d_mc_rel=d_mc_rel, d_tc=d_tc))
        if s + 1 < len(stages):
            cur = refine(cur, idx, r, d_mc_rel, d_tc)
            d_mc_rel /= r
            d_tc /= r
    return out
