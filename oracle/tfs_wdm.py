"""CPU fp64 oracle for the statistic in a real-coefficient orthonormal wavelet (WDM) pixel basis.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  It shares no code with the
CUDA path (``paper_2510_19047_b200``) and imports nothing from it.

Why it exists.  BASELINE.json's north_star speaks of "wavelet-pixel" data in an "orthonormal TF basis";
the paper itself works on complex short-time Fourier tranches (Eq. 16) and points to
wavelet time-frequency methods only as related work (P:27 refs [28, 49]; P:297 refs [28, 69]).  The basis
equations live in ref. [28], which is NOT in the container, so everything below is written from the
standard Wilson-Daubechies-Meyer construction and every choice is a numbered reading:

  W1  grid: Nt time pixels x Nf frequency layers, N = Nt Nf real samples at cadence dt, pixel duration
      DT = Nf dt, layer spacing DF = 1/(2 DT): critically sampled, Nt Nf real coefficients.
  W2  window: Meyer-type frequency response with the roll-off spread over the whole layer spacing,
      Phi(omega) = cos(pi |omega| / (2 DOmega)) / sqrt(DOmega) for |omega| <= DOmega = 2 pi DF, else 0
      (it satisfies Phi(w)^2 + Phi(w - DOmega)^2 = 1/DOmega; the family's steepness parameter is fixed at
      "no flat top": this makes a pixel overlap only its two neighbouring layers and gives the chirp
      response below a closed form in Fresnel integrals).
  W3  basis functions (k = sample index, phi[k] the window centred at k = 0, sum phi^2 = 1):
        0 < m < Nf, n + m even:  g_nm[k] = sqrt2 (-1)^(n m) cos(pi m k / Nf) phi[k - n Nf]
        0 < m < Nf, n + m odd :  g_nm[k] = sqrt2            sin(pi m k / Nf) phi[k - n Nf]
        m = 0  (n even)       :  g_n0[k] = phi[k - n Nf]
        m = Nf (n + Nf even)  :  g_nNf[k] = (-1)^k phi[k - n Nf]
      The Nyquist layer is stored in the unused slots of column 0 (column 0 of row n holds the DC layer
      when n is even and the Nyquist layer of time n - 1 + (Nf odd) ... see ``edge_slot``).
  W4  template pixel of a chirp h(t) = A cos Phi(t): phase expanded to second order about the pixel centre
      t_n = n DT (the paper's Eqs. 12-15 moved to the pixel centre), amplitude frozen; then
        H_nm = eps_nm (A_n / sqrt2) exp(i Phi_n) K(x, kappa),   x = f_n/DF - m,  kappa = 4 fdot_n DT^2,
        eps = 1 (n + m even), i (-1)^(n m) (n + m odd),
        K(x, kappa) = exp(i pi/4) / sqrt(kappa) * int_{-1}^{1} cos(pi y/2) exp(-i pi (y + x)^2 / kappa) dy
      (the window's response to a linear chirp; kappa -> 0: cos(pi x/2) on |x| < 1; the common factor
      1/sqrt(DOmega) is dropped on both sides).  Re H is the pixel of the chirp at phase offset 0 and
      Im H that at -pi/2: a template of any phase is cos(p) Re H - sin(p) Im H.
  W5  layer window: m in [ceil(x_f) - 1 - Hw, floor(x_f) + 1 + Hw] with x_f = f_n / DF (the two layers the
      track sits between, plus Hw on either side, default 2), clipped to [1, Nf - 1].
  W6  statistic per segment: data are real, so the two template quadratures are not exactly orthogonal;
      P_n = max over amplitude and phase of the segment's log-likelihood = [a b] G^-1 [a b]^T with
      a + i b = sum_alpha sum W d (T_alpha H) and G the 2 x 2 Gram matrix of (Re, Im)(T_alpha H) under W
      (Eq. 5 and P:104: each segment is maximised over two parameters).  Upsilon = sum_n P_n.
  W7  activity: pixel n is used when tau_n = tc - t_n > 2 DT (the window reaches about one pixel on either
      side of its centre), f_lo <= f_n, f_n + |fdot_n| DT <= f_hi, kappa <= kappa_max; gaps as P:297.

Pins: tests/test_wdm_pins.py (orthonormality of the complete basis, reconstruction, Parseval, tones land in
two layers, the chirp response against the exact transform of a sampled chirp and against its kappa -> 0
limit, noiseless injection Upsilon_N = rho^2, noise-only mean 2 N, recovery of a time-domain 0PN chirp).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

MTSUN_S = 4.925490947e-6
YEAR_S = 365.25 * 86400.0


@dataclass(frozen=True)
class WdmGrid:
    Nt: int
    Nf: int
    dt: float

    @property
    def DT(self) -> float:
        return self.Nf * self.dt

    @property
    def DF(self) -> float:
        return 1.0 / (2.0 * self.DT)

    @property
    def N(self) -> int:
        return self.Nt * self.Nf


@dataclass(frozen=True)
class WdmOpts:
    half_width: int = 2           # Hw (W5)
    kappa_max: float = 8.0        # pixels with 4 fdot DT^2 above this are skipped (W7)
    f_lo: float | None = None
    f_hi: float | None = None

    def band(self, g: WdmGrid):
        lo = g.DF if self.f_lo is None else self.f_lo
        hi = (g.Nf - 1) * g.DF if self.f_hi is None else self.f_hi
        return lo, hi


# ----------------------------------------------------------------------------------------------
# W2: the window, W3: the basis
# ----------------------------------------------------------------------------------------------
def window(g: WdmGrid):
    """phi[k], k = 0..N-1 (periodic, centred at k = 0), sum phi^2 = 1: the inverse DFT of
    Phi[l] = sqrt(2 Nf) cos(pi l / Nt) on |l| <= Nt/2 (DFT bin l <-> omega = 2 pi l / (N dt); DOmega <-> Nt/2 bins)."""
    if g.Nt % 2:
        raise ValueError("Nt must be even")
    N, half = g.N, g.Nt // 2
    Phi = np.zeros(N)
    l = np.arange(-half, half + 1)
    Phi[l % N] = math.sqrt(2.0 * g.Nf) * np.cos(math.pi * l / g.Nt)
    return np.fft.ifft(Phi).real


def edge_slot(n: int, g: WdmGrid):
    """Which basis function column 0 of row n holds: ('dc', n) for even n; ('nyq', n') with n' the Nyquist
    layer's time index stored there, n' = n - 1 if Nf is even (n' even) else n (n' odd)."""
    if n % 2 == 0:
        return "dc", n
    return "nyq", (n - 1 if g.Nf % 2 == 0 else n)


def basis_function(n: int, m: int, g: WdmGrid, phi=None):
    """g_nm[k] (W3) for the storage slot (n, m), m = 0..Nf-1."""
    phi = window(g) if phi is None else phi
    k = np.arange(g.N)
    if m == 0:
        kind, nn = edge_slot(n, g)
        sh = np.roll(phi, nn * g.Nf)
        return sh if kind == "dc" else ((-1.0) ** k) * sh
    sh = np.roll(phi, n * g.Nf)
    if (n + m) % 2 == 0:
        return math.sqrt(2.0) * (-1.0) ** (n * m) * np.cos(math.pi * m * k / g.Nf) * sh
    return math.sqrt(2.0) * np.sin(math.pi * m * k / g.Nf) * sh


def transform_direct(x, g: WdmGrid):
    """w[n][m] = sum_k x[k] g_nm[k], written out (O(N^2))."""
    x = np.asarray(x, dtype=np.float64)
    phi = window(g)
    w = np.zeros((g.Nt, g.Nf))
    for n in range(g.Nt):
        for m in range(g.Nf):
            w[n, m] = np.dot(x, basis_function(n, m, g, phi))
    return w


def inverse_direct(w, g: WdmGrid):
    """x[k] = sum_nm w[n][m] g_nm[k] (the basis is orthonormal)."""
    phi = window(g)
    x = np.zeros(g.N)
    for n in range(g.Nt):
        for m in range(g.Nf):
            x += w[n, m] * basis_function(n, m, g, phi)
    return x


def transform(x, g: WdmGrid):
    """The same coefficients through FFTs: with X = DFT(x),
    y_m[n] = sum_k x[k] phi[k - n Nf] exp(-i pi m k / Nf) = (1/N) sum_{|l| <= Nt/2} X[m Nt/2 + l] Phi[l] exp(2 pi i l n / Nt),
    and the cosine / sine pixels are sqrt2 (-1)^(nm) Re y, -sqrt2 Im y (pinned against transform_direct)."""
    x = np.asarray(x, dtype=np.float64)
    N, Nt, Nf, half = g.N, g.Nt, g.Nf, g.Nt // 2
    X = np.fft.fft(x)
    l = np.arange(-half, half + 1)
    Phi = math.sqrt(2.0 * Nf) * np.cos(math.pi * l / Nt)
    n = np.arange(Nt)
    ph = np.exp(2j * math.pi * np.outer(n, l) / Nt)                       # [Nt][Nt+1]
    w = np.zeros((Nt, Nf))
    for m in range(0, Nf + 1):
        y = ph @ (X[(m * half + l) % N] * Phi) / N                        # y_m[n]
        if m == 0:
            w[0::2, 0] = y.real[0::2]
        elif m == Nf:
            nn = n[(n + Nf) % 2 == 0]
            slot = nn + 1 if Nf % 2 == 0 else nn
            w[slot, 0] = y.real[nn]
        else:
            even = (n + m) % 2 == 0
            w[even, m] = math.sqrt(2.0) * ((-1.0) ** (n[even] * m)) * y.real[even]
            w[~even, m] = -math.sqrt(2.0) * y.imag[~even]
    return w


# ----------------------------------------------------------------------------------------------
# W4: response of the window to a linear chirp
# ----------------------------------------------------------------------------------------------
def chirp_response_closed(x, kappa):
    """K(x, kappa) in closed form: completing the square in the exponent of each half of cos(pi y/2) turns the
    defining integral (W4) into Fresnel integrals F = C + i S (oracle/tfs_oracle.py's own routine),
        K = exp(i pi/4)/(2 sqrt2) sum_{s=+-1} exp(i pi kappa/16 - s i pi x/2) conj[F(v_hi) - F(v_lo)],
        v_hi,lo = sqrt(2/kappa) (x +- 1 - s kappa/4).
    Pinned against the quadrature below where both are affordable (tests/test_wdm_pins.py)."""
    from oracle.tfs_oracle import fresnel_cs
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    tot = np.zeros(x.shape, dtype=np.complex128)
    for s in (+1.0, -1.0):
        vhi = math.sqrt(2.0 / kappa) * (x + 1.0 - s * kappa / 4.0)
        vlo = math.sqrt(2.0 / kappa) * (x - 1.0 - s * kappa / 4.0)
        Ch, Sh = fresnel_cs(vhi)
        Cl, Sl = fresnel_cs(vlo)
        tot += np.exp(1j * (math.pi * kappa / 16.0 - s * 0.5 * math.pi * x)) * np.conj((Ch - Cl) + 1j * (Sh - Sl))
    return tot * np.exp(0.25j * math.pi) / (2.0 * math.sqrt(2.0))


KAPPA_QUADRATURE_MIN = 0.02      # below this the quadrature needs > 1e4 panels per pixel: the closed form takes over


def chirp_response(x, kappa, panels_per_cycle: int = 6):
    """K(x, kappa): Gauss-Legendre quadrature of its defining integral (W4) for kappa >= KAPPA_QUADRATURE_MIN, the
    closed form (pinned against the quadrature) for slower chirps; kappa <= 1e-9: the limit cos(pi x/2)."""
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    out = np.empty(x.shape, dtype=np.complex128)
    if kappa <= 1e-9:
        out[:] = np.where(np.abs(x) < 1.0, np.cos(0.5 * math.pi * x), 0.0)
        return out
    if kappa < KAPPA_QUADRATURE_MIN:
        return chirp_response_closed(x, kappa)
    xs, ws = np.polynomial.legendre.leggauss(16)
    for i, xv in enumerate(x.ravel()):
        # the phase pi (y + x)^2 / kappa turns at most 2 (|x| + 1) / kappa times per unit y
        rate = 2.0 * (abs(xv) + 1.0) / kappa + 1.0
        npan = int(math.ceil(2.0 * rate * panels_per_cycle)) + 2
        edges = np.linspace(-1.0, 1.0, npan + 1)
        mid = 0.5 * (edges[1:] + edges[:-1])
        hw = 0.5 * (edges[1:] - edges[:-1])
        y = (mid[:, None] + hw[:, None] * xs[None, :])
        val = np.cos(0.5 * math.pi * y) * np.exp(-1j * math.pi * (y + xv) ** 2 / kappa)
        out.ravel()[i] = np.sum(val * ws[None, :] * hw[:, None])
    return out * np.exp(0.25j * math.pi) / math.sqrt(kappa)


# ----------------------------------------------------------------------------------------------
# track at the pixel centres and the dense template
# ----------------------------------------------------------------------------------------------
def track(Mc_msun, tc, phic, amp, g: WdmGrid, o: WdmOpts, gap_mask=None):
    """0PN track at the pixel centres t_n = n DT (textbook closed form as in oracle/tfs_oracle.py)."""
    n = np.arange(g.Nt, dtype=np.float64)
    DT, DF = g.DT, g.DF
    M = Mc_msun * MTSUN_S
    tau = tc - n * DT
    ok = tau > 2.0 * DT
    if gap_mask is not None:
        ok = ok & (np.asarray(gap_mask) != 0)
    ok = ok & np.isfinite(tau)
    tau_s = np.where(ok, tau, 1.0)
    X = tau_s / (5.0 * M)
    f = X ** (-0.375) / (8.0 * math.pi * M)
    phi = phic - 2.0 * X ** 0.625
    fdot = 3.0 * f / (8.0 * tau_s)
    A = amp * f ** (2.0 / 3.0)
    xf = f / DF
    kappa = 4.0 * fdot * DT * DT
    f_lo, f_hi = o.band(g)
    active = ok & (f >= f_lo) & (f + fdot * DT <= f_hi) & (kappa <= o.kappa_max)
    m_lo = np.clip(np.ceil(xf) - 1 - o.half_width, 1, g.Nf - 1).astype(np.int64)
    m_hi = np.clip(np.floor(xf) + 1 + o.half_width, 1, g.Nf - 1).astype(np.int64)
    return dict(active=active, f=f, fdot=fdot, phi=phi, A=A, xf=xf, kappa=kappa, m_lo=m_lo, m_hi=m_hi)


def eps(n, m):
    """eps_nm of W4."""
    n = np.asarray(n, dtype=np.int64)
    m = np.asarray(m, dtype=np.int64)
    odd = (n + m) % 2 == 1
    return np.where(odd, 1j * (-1.0) ** ((n * m) % 2), 1.0 + 0j)


def dense_template(Mc_msun, tc, phic, amp, g: WdmGrid, o: WdmOpts, gap_mask=None, truncate=True):
    """Dense [Nt][Nf] complex128 template H (W4), zero outside each pixel's layer window (all layers
    1..Nf-1 of every active pixel when truncate = False)."""
    tr = track(Mc_msun, tc, phic, amp, g, o, gap_mask)
    H = np.zeros((g.Nt, g.Nf), dtype=np.complex128)
    for n in np.nonzero(tr["active"])[0]:
        lo, hi = (tr["m_lo"][n], tr["m_hi"][n]) if truncate else (1, g.Nf - 1)
        if not truncate:
            # K vanishes (to quadrature accuracy) far from the track: fill only where it can matter
            lo = max(1, int(math.floor(tr["xf"][n] - 3 - 2 * tr["kappa"][n])))
            hi = min(g.Nf - 1, int(math.ceil(tr["xf"][n] + 3 + 2 * tr["kappa"][n])))
        m = np.arange(lo, hi + 1)
        K = chirp_response(tr["xf"][n] - m, tr["kappa"][n])
        H[n, lo:hi + 1] = eps(n, m) * (tr["A"][n] / math.sqrt(2.0)) * np.exp(1j * tr["phi"][n]) * K
    return H


def segment_products(H, T, D, W, gap_mask, N_seg: int):
    """Per segment: a + i b = sum_alpha sum W d (T_alpha H), and the Gram matrix entries
    (hcc, hss, hcs) = sum_alpha sum W (Re^2, Im^2, Re Im)(T_alpha H), dense sums over every pixel (W6)."""
    Cn, Nt, Nf = D.shape
    gm = np.ones(Nt) if gap_mask is None else (np.asarray(gap_mask) != 0).astype(np.float64)
    seg = (np.arange(Nt, dtype=np.int64) * N_seg) // Nt
    z = np.zeros(N_seg, dtype=np.complex128)
    G = np.zeros((N_seg, 3))
    for a in range(Cn):
        Wa = np.ones((Nt, Nf)) if W is None else W[a].astype(np.float64)
        Y = T[a] * H
        za = np.sum(Wa * D[a] * Y, axis=1) * gm
        z += np.bincount(seg, weights=za.real, minlength=N_seg) + 1j * np.bincount(seg, weights=za.imag, minlength=N_seg)
        for j, q in enumerate((Y.real ** 2, Y.imag ** 2, Y.real * Y.imag)):
            G[:, j] += np.bincount(seg, weights=np.sum(Wa * q, axis=1) * gm, minlength=N_seg)
    return z, G


def combine(z, G):
    """P_n = [a b] G^-1 [a b]^T (0 where the Gram matrix is singular); Upsilon = sum P_n (W6)."""
    a, b = z.real, z.imag
    hcc, hss, hcs = G[:, 0], G[:, 1], G[:, 2]
    det = hcc * hss - hcs * hcs
    with np.errstate(divide="ignore", invalid="ignore"):
        P = np.where(det > 0, (a * a * hss - 2.0 * a * b * hcs + b * b * hcc) / det, 0.0)
    return P, float(np.sum(P))


def evaluate(params, D, W, gap_mask, g: WdmGrid, N_seg: int, o: WdmOpts = WdmOpts()):
    """Upsilon of every row of params [n][8] (columns as in include/tfs.h) on real WDM data D [C][Nt][Nf].
    Returns dict(upsilon[n], seg_power[n][N_seg], seg_dh[n][N_seg] complex (a + i b), seg_gram[n][N_seg][3])."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    n = params.shape[0]
    ups = np.zeros(n)
    segP = np.zeros((n, N_seg))
    segz = np.zeros((n, N_seg), dtype=np.complex128)
    segG = np.zeros((n, N_seg, 3))
    for i in range(n):
        p = params[i]
        if not np.all(np.isfinite(p)) or p[0] <= 0:
            continue
        H = dense_template(p[0], p[1], p[2], p[7], g, o, gap_mask, truncate=True)
        T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6], 0.0])
        z, G = segment_products(H, T[: D.shape[0]], D, W, gap_mask, N_seg)
        P, U = combine(z, G)
        ups[i], segP[i], segz[i], segG[i] = U, P, z, G
    return dict(upsilon=ups, seg_power=segP, seg_dh=segz, seg_gram=segG)


def injection(p, rho: float, W, gap_mask, g: WdmGrid, o: WdmOpts = WdmOpts(), phase: float = 0.0, truncate=True):
    """Real WDM-domain signal of parameters p at phase offset `phase`, per channel,
    s_alpha = Re(T_alpha exp(i phase) H), scaled so that sum_alpha sum W s^2 = rho^2 over the valid pixels."""
    H = dense_template(p[0], p[1], p[2], p[7], g, o, None, truncate=truncate)
    T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6], 0.0])
    Cn = 2 if W is None else W.shape[0]
    S = np.stack([(T[a] * np.exp(1j * phase) * H).real for a in range(Cn)])
    gm = np.ones(g.Nt) if gap_mask is None else (np.asarray(gap_mask) != 0).astype(np.float64)
    Wd = np.ones_like(S) if W is None else W.astype(np.float64)
    S *= rho / math.sqrt(float(np.sum(Wd * S * S * gm[None, :, None])))
    return S * gm[None, :, None]
