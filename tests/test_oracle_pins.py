"""Pins for the CPU oracle (oracle/tfs_oracle.py) against what the paper and mathematics fix.

None of these call the CUDA path.  Pin ids P1..P12 follow DESIGN.md section 5 / SURVEY.md 8(c).
"""
import cmath
import math
import os

import numpy as np
import pytest

from oracle import tfs_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
TINY = O.Grid(512, 1024, 5.0)
SMALL = O.Grid(128, 256, 5.0)       # DT = 2560 s
# cfg1 injection (BASELINE.json configs[0]): Mc 30, tc 1 yr, antenna weights (0.7, 0.5)
INJ = np.array([30.0, 1.0 * O.YEAR_S, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])


def _gl(fun, a, b, n=64):
    """Gauss-Legendre quadrature of fun over [a, b]."""
    xs, ws = np.polynomial.legendre.leggauss(n)
    t = 0.5 * (b - a) * xs + 0.5 * (b + a)
    return 0.5 * (b - a) * np.sum(ws * fun(t))


# ------------------------------------------------------------------------------------------
# P1  Fresnel integrals
# ------------------------------------------------------------------------------------------
def test_p1_fresnel_printed_values():
    for line in open(os.path.join(GOLD, "fresnel_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        z, c, s = line.split()
        tol = 0.6 * 10.0 ** (-len(c.split(".")[1]))
        C, S = O.fresnel_cs(np.array([float(z)]))
        assert abs(C[0] - float(c)) < tol and abs(S[0] - float(s)) < tol, (z, C, S)


def test_p1_fresnel_definition_by_quadrature():
    # the defining integrals, panel by panel, |z| up to 12 (crosses series/CF switch)
    edges = np.linspace(0.0, 12.0, 481)
    Cq = np.cumsum([_gl(lambda x: np.cos(0.5 * np.pi * x * x), a, b, 24) for a, b in zip(edges[:-1], edges[1:])])
    Sq = np.cumsum([_gl(lambda x: np.sin(0.5 * np.pi * x * x), a, b, 24) for a, b in zip(edges[:-1], edges[1:])])
    C, S = O.fresnel_cs(edges[1:])
    assert np.max(np.abs(C - Cq)) < 1e-12 and np.max(np.abs(S - Sq)) < 1e-12


def test_p1_fresnel_increments_large_argument():
    # C(b)-C(a) = int_a^b cos(pi x^2/2) dx for narrow intervals at large z (v reaches ~1e3 for slow chirps)
    rng = np.random.default_rng(0)
    for z in [7.3, 20.1, 77.7, 300.2, 1500.4]:
        a = z + rng.uniform(0, 1)
        b = a + 0.5 / z
        Ca, Sa = O.fresnel_cs(np.array([a]))
        Cb, Sb = O.fresnel_cs(np.array([b]))
        assert abs((Cb - Ca)[0] - _gl(lambda x: np.cos(0.5 * np.pi * x * x), a, b)) < 2e-13
        assert abs((Sb - Sa)[0] - _gl(lambda x: np.sin(0.5 * np.pi * x * x), a, b)) < 2e-13


def test_p1_fresnel_symmetry_limits_asymptote():
    z = np.linspace(0.0, 40.0, 4001)
    C, S = O.fresnel_cs(z)
    Cm, Sm = O.fresnel_cs(-z)
    assert np.array_equal(C, -Cm) and np.array_equal(S, -Sm)           # odd
    Ci, Si = O.fresnel_cs(np.array([np.inf, -np.inf, 1e9]))
    assert np.allclose(Ci, [0.5, -0.5, 0.5], atol=1e-9) and np.allclose(Si, [0.5, -0.5, 0.5], atol=1e-9)
    # leading asymptote (the paper's Eqs. 23-24) with the next term 1/(pi^2 z^3) as the bound
    zz = z[z > 6]
    C, S = O.fresnel_cs(zz)
    ph = 0.5 * np.pi * zz * zz
    bound = 1.02 / (np.pi ** 2 * zz ** 3)
    assert np.all(np.abs(C - (0.5 + np.sin(ph) / (np.pi * zz))) <= bound)
    assert np.all(np.abs(S - (0.5 - np.cos(ph) / (np.pi * zz))) <= bound)


def test_p1_fresnel_vs_libraries():
    from scipy.special import fresnel
    z = np.concatenate([np.linspace(-9, 9, 3001), np.geomspace(9, 3000, 500)])
    S0, C0 = fresnel(z)
    C, S = O.fresnel_cs(z)
    assert np.max(np.abs(C - C0)) < 1e-12 and np.max(np.abs(S - S0)) < 1e-12
    mp = pytest.importorskip("mpmath")
    for x in [0.3, 1.9, 2.1, 4.7, 33.3]:
        C, S = O.fresnel_cs(np.array([x]))
        assert abs(C[0] - float(mp.fresnelc(x))) < 1e-13 and abs(S[0] - float(mp.fresnels(x))) < 1e-13


def test_p1_paper_approximants_error_level():
    # DESIGN.md C8: the printed Eqs. 25-28 reach ~2.2e-3, not the claimed 1e-4
    z = np.linspace(-6, 6, 120001)
    Cp, Sp = O.fresnel_cs_paper(z)
    Ce, Se = O.fresnel_cs(z)
    eC, eS = np.max(np.abs(Cp - Ce)), np.max(np.abs(Sp - Se))
    assert 1.9e-3 < eC < 2.3e-3 and 2.0e-3 < eS < 2.4e-3
    z = np.array([6.0 + 1e-9])                                         # Eqs. 23-24 just above the switch
    e = np.abs(np.array(O.fresnel_cs_paper(z)) - np.array(O.fresnel_cs(z))).max()
    assert 3e-4 < e < 6e-4
    z = np.linspace(6.001, 60, 5000)                                   # and they are odd-extended
    assert np.allclose(O.fresnel_cs_paper(-z)[0], -O.fresnel_cs_paper(z)[0])


# ------------------------------------------------------------------------------------------
# P2  Eq. 16: sign, phase, normalisation
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c", [1e-4, 3e-2, 0.5, 3.0, 25.0, 150.0])
def test_p2_kernel_is_fourier_integral_of_linear_chirp(c):
    # h~(f_k)/DT = int_0^1 A exp{i(phi + 2 pi u s + pi c s^2)} ds, u = x - k  (Eq. 16 is this
    # integral in closed form).  Direct quadrature, independent of Fresnel functions.
    x, phi, A = 200.37, 0.83, 1.7
    k = np.arange(150, 420)
    Hk = O.kernel_pixels(x, c, phi, A, k)
    for kk, h in zip(k[::17], Hk[::17]):
        u = x - kk
        npan = int(8 + 2 * (abs(u) + c))
        e = np.linspace(0, 1, npan + 1)
        q = sum(_gl(lambda s: np.exp(1j * (phi + 2 * np.pi * u * s + np.pi * c * s * s)), a, b, 32)
                for a, b in zip(e[:-1], e[1:]))
        # literal Eq. 16 in fp64: the phase pi v^2/2 of v ~ u sqrt(2/c) loses ~1e-16 v^2 rad
        assert abs(h - A * q) < 1e-10 + 1.5e-13 / c


@pytest.mark.parametrize("c", [1e-4, 0.5, 3.0, 25.0, 150.0])
def test_p2_kernel_vs_fft_of_sampled_chirp(c):
    # sampled chirp in one tranche of the Tiny grid: dt*FFT[k] (time origin at tranche start)
    g = TINY
    N = 2 * g.Nf
    x, phi, A = 300.37, 1.1, 1.0
    f, fdot = x * g.df, c * g.df / g.DT
    t = np.arange(N) * g.dt
    xt = A * np.exp(1j * (phi + 2 * np.pi * f * t + np.pi * fdot * t * t))
    X = g.dt * np.fft.fft(xt)[: g.Nf] / g.DT
    Hk = O.kernel_pixels(x, c, phi, A, np.arange(g.Nf))
    peak = np.max(np.abs(Hk))
    # left Riemann sum vs integral: endpoint term (dt/2)(x(0) - x(DT)), |.| <= A/N
    assert np.max(np.abs(X - Hk)) < 1.05 * A / N
    if c <= 3.0:
        assert np.max(np.abs(X - Hk)) < 3e-3 * peak
    # trapezoid-corrected sum (exp(-2 pi i f_k DT) = 1): error drops to O(1/N^2)
    xT = A * np.exp(1j * (phi + 2 * np.pi * f * g.DT + np.pi * fdot * g.DT ** 2))
    Xt = X + 0.5 * (xT - xt[0]) / N
    u = x - np.arange(g.Nf)                                            # Euler-Maclaurin: h^2/12 [F'(1)-F'(0)]
    bound = 1.1 * A * 2 * np.pi * (np.abs(u) + np.abs(u + c)) / (12.0 * N * N) + 1e-6
    assert np.all(np.abs(Xt - Hk) < bound)


def test_p2_slow_chirp_limit_is_sinc():
    # c -> 0: int_0^1 exp(2 pi i u s) ds = exp(i pi u) sin(pi u)/(pi u)  (textbook)
    x, phi, A, c = 57.3, -0.4, 2.0, 1e-7
    k = np.arange(40, 75)
    u = x - k
    ref = A * np.exp(1j * (phi + np.pi * u)) * np.sinc(u)
    assert np.max(np.abs(O.kernel_pixels(x, c, phi, A, k) - ref)) < 1e-6


# ------------------------------------------------------------------------------------------
# P3  Parseval
# ------------------------------------------------------------------------------------------
def test_p3_block_dft_parseval():
    g = TINY
    rng = np.random.default_rng(3)
    N = 2 * g.Nf
    x = rng.standard_normal((16, N))
    X = g.dt * np.fft.rfft(x, axis=1)                                   # bins 0..Nf
    lhs = (2 * np.sum(np.abs(X[:, 1:-1]) ** 2) + np.sum(np.abs(X[:, 0]) ** 2) + np.sum(np.abs(X[:, -1]) ** 2)) * g.df
    rhs = np.sum(x * x) * g.dt
    assert abs(lhs / rhs - 1) < 1e-12


def test_p3_template_norm_matches_time_domain():
    # TF-domain <h|h> of the dense untruncated template vs the time-domain norm of A(t)e^{i phi(t)}
    g, o = TINY, O.Opts()
    Hd = O.dense_template(INJ[0], INJ[1], INJ[2], INJ[7], g, o, truncate=False)
    tf_norm = np.sum(np.abs(Hd) ** 2) * g.DT                            # sum |h~|^2 df, h~ = H*DT
    t = (np.arange(g.Nt * 2 * g.Nf) + 0.5) * g.dt
    M = INJ[0] * O.MTSUN_S
    ft = ((INJ[1] - t) / (5 * M)) ** (-0.375) / (8 * np.pi * M)
    td_norm = np.sum((INJ[7] * ft ** (2.0 / 3.0)) ** 2) * g.dt
    assert abs(tf_norm / td_norm - 1) < 1e-3


# ------------------------------------------------------------------------------------------
# helpers: small noisy data set
# ------------------------------------------------------------------------------------------
def _noise(g, seed, C=2):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((C, g.Nt, g.Nf)) + 1j * rng.standard_normal((C, g.Nt, g.Nf))


def _weights(g, seed, C=2):
    rng = np.random.default_rng(seed + 77)
    return rng.uniform(0.3, 2.0, (C, g.Nt, g.Nf))


SMALL_T = np.array([30.0, 0.12 * O.YEAR_S, 1.0, 0.6, 0.3, -0.2, 0.5, 1.3])   # chirps out inside SMALL's span? no: tc > Tobs


# ------------------------------------------------------------------------------------------
# P4  N_seg = 1 is the phase-maximised coherent SNR^2
# ------------------------------------------------------------------------------------------
def test_p4_nseg1_is_phase_maximised_snr2():
    g, o = SMALL, O.Opts()
    D, W = _noise(g, 1), _weights(g, 1)
    D = D + O.injection(SMALL_T, 6.0, W, None, g, o)
    res = O.evaluate(SMALL_T[None], D, W, None, g, 1, o)
    Hd = O.dense_template(*SMALL_T[[0, 1, 2, 7]], g, o)
    T = [SMALL_T[3] + 1j * SMALL_T[4], SMALL_T[5] + 1j * SMALL_T[6]]
    best = 0.0
    for phi in np.linspace(0, 2 * np.pi, 3600, endpoint=False):
        num = den = 0.0
        for a in range(2):
            y = T[a] * Hd * np.exp(1j * phi)
            num += np.sum(W[a] * (D[a].real * y.real + D[a].imag * y.imag))   # <d|y> as a real inner product
            den += np.sum(W[a] * (y.real ** 2 + y.imag ** 2))
        best = max(best, num * abs(num) / den)                          # rho^2 with the sign of rho
    assert abs(best / res["upsilon"][0] - 1) < 1e-6


# ------------------------------------------------------------------------------------------
# P5  noiseless injection at the true parameters: Upsilon_N = rho^2 for every N
# ------------------------------------------------------------------------------------------
def test_p5_noiseless_injection_gives_rho2():
    g, o = TINY, O.Opts()
    rho = 20.0
    S = O.injection(INJ, rho, None, None, g, o, truncate=True)
    for N in (1, 4, 16, 64):
        r = O.evaluate(INJ[None], S, None, None, g, N, o)
        assert abs(r["upsilon"][0] / rho ** 2 - 1) < 1e-10
        assert np.allclose(np.sum(r["seg_hh"]) * (rho ** 2 / np.sum(r["seg_hh"])), rho ** 2)
    # untruncated injection, truncated search template: the 21-bin window keeps ~99 %
    S = O.injection(INJ, rho, None, None, g, o, truncate=False)
    r = O.evaluate(INJ[None], S, None, None, g, 4, o)
    assert 0.975 < r["upsilon"][0] / rho ** 2 < 0.999


# ------------------------------------------------------------------------------------------
# P6  time-domain injection (real chirp -> per-tranche FFT) is recovered within 2 % in SNR
# ------------------------------------------------------------------------------------------
def test_p6_time_domain_injection_recovery():
    g, o = TINY, O.Opts()
    N = 2 * g.Nf
    t = np.arange(g.Nt * N) * g.dt
    M = INJ[0] * O.MTSUN_S
    X = (INJ[1] - t) / (5 * M)
    f = X ** (-0.375) / (8 * np.pi * M)
    h = INJ[7] * f ** (2.0 / 3.0) * np.exp(1j * (INJ[2] - 2 * X ** 0.625))       # A(t) e^{i phi(t)} (Eq. 11)
    T = [INJ[3] + 1j * INJ[4], INJ[5] + 1j * INJ[6]]
    D = np.empty((2, g.Nt, g.Nf), dtype=np.complex128)
    rho2_td = 0.0
    for a in range(2):
        s = (T[a] * h).real                                              # real TDI strain
        D[a] = (np.fft.rfft(s.reshape(g.Nt, N), axis=1) / N)[:, : g.Nf]  # = dt*FFT/DT
        rho2_td += np.sum(s * s) / (2 * N)                               # sum_{k>0} |X_k|^2 by Parseval
    for Nseg in (1, 4):
        r = O.evaluate(INJ[None], D, None, None, g, Nseg, o)
        # template is the analytic signal, data the real one: <d|y> picks up 1/2 (C16): compare SNR^2
        assert math.sqrt(r["upsilon"][0] / rho2_td) > 0.98
        assert r["upsilon"][0] / rho2_td < 1.0 + 1e-9


# ------------------------------------------------------------------------------------------
# P7  noise only: each segment term is chi^2_2  =>  E[Upsilon] = 2 N_eff, Var = 4 N_eff
# ------------------------------------------------------------------------------------------
def test_p7_noise_only_expectation():
    g, o = O.Grid(64, 128, 5.0), O.Opts()
    nseed = 10000
    Hd = O.dense_template(*SMALL_T[[0, 1, 2, 7]], g, o)
    T = np.array([SMALL_T[3] + 1j * SMALL_T[4], SMALL_T[5] + 1j * SMALL_T[6]])
    W = _weights(g, 5)
    sig = 1.0 / np.sqrt(W)                                               # E|D|^2 = 2/W
    ups = {N: np.empty(nseed) for N in (1, 4, 16)}
    for s in range(nseed):
        D = _noise(g, 10_000 + s) * sig
        for N in ups:
            z, hh = O.segment_products(Hd, T, D, W, None, N)
            ups[N][s] = O.combine(z, hh)[1]
    for N, u in ups.items():
        assert abs(u.mean() - 2 * N) < 3 * 2 * math.sqrt(N / nseed), (N, u.mean())
        assert abs(u.var() / (4 * N) - 1) < 0.08
    # a single segment term is chi^2_2: P(P_n > x) = exp(-x/2)
    assert abs(np.mean(ups[1] > 4.0) - math.exp(-2.0)) < 0.012


# ------------------------------------------------------------------------------------------
# P8  refinement can only raise the statistic (Cauchy-Schwarz), P9 invariances
# ------------------------------------------------------------------------------------------
def test_p8_monotone_under_refinement():
    g, o = SMALL, O.Opts()
    D, W = _noise(g, 8), _weights(g, 8)
    rng = np.random.default_rng(8)
    P = np.tile(SMALL_T, (6, 1))
    P[:, 0] = rng.uniform(20, 60, 6)
    P[:, 1] = rng.uniform(0.05, 3.0, 6) * O.YEAR_S
    prev = None
    for N in (1, 2, 4, 8, 16, 32, 64, 128):
        u = O.evaluate(P, D, W, None, g, N, o)["upsilon"]
        if prev is not None:
            assert np.all(u >= prev * (1 - 1e-12))
        prev = u


def test_p9_invariances():
    g, o = SMALL, O.Opts()
    D, W = _noise(g, 9), _weights(g, 9)
    base = O.evaluate(SMALL_T[None], D, W, None, g, 4, o)
    u0 = base["upsilon"][0]
    p = SMALL_T.copy(); p[2] += 1.234                                   # phic
    assert abs(O.evaluate(p[None], D, W, None, g, 4, o)["upsilon"][0] / u0 - 1) < 1e-10
    p = SMALL_T.copy(); p[7] *= 3.7                                     # amp
    r = O.evaluate(p[None], D, W, None, g, 4, o)
    assert abs(r["upsilon"][0] / u0 - 1) < 1e-10
    assert np.allclose(r["seg_hh"], 3.7 ** 2 * base["seg_hh"], rtol=1e-12)
    p = SMALL_T.copy()                                                   # common phase of (T_A, T_E)
    rot = cmath.exp(0.77j)
    ta, te = (p[3] + 1j * p[4]) * rot, (p[5] + 1j * p[6]) * rot
    p[3:7] = ta.real, ta.imag, te.real, te.imag
    assert abs(O.evaluate(p[None], D, W, None, g, 4, o)["upsilon"][0] / u0 - 1) < 1e-10
    assert abs(O.evaluate(SMALL_T[None], 2.5 * D, W, None, g, 4, o)["upsilon"][0] / (6.25 * u0) - 1) < 1e-10
    assert abs(O.evaluate(SMALL_T[None], D, 1.7 * W, None, g, 4, o)["upsilon"][0] / (1.7 * u0) - 1) < 1e-10


# ------------------------------------------------------------------------------------------
# P10 gaps
# ------------------------------------------------------------------------------------------
def test_p10_gaps():
    g, o = TINY, O.Opts()
    rho = 20.0
    S = O.injection(INJ, rho, None, None, g, o, truncate=True)
    rng = np.random.default_rng(10)
    gap = (rng.random(g.Nt) > 0.15).astype(np.uint8)
    p_lost = 1.0 - gap.mean()
    r = O.evaluate(INJ[None], S, None, gap, g, 1, o)
    # nearly monochromatic: Upsilon_1 drops by the lost fraction (~15 % at 85 % duty cycle)
    assert abs((1 - r["upsilon"][0] / rho ** 2) - p_lost) < 0.01
    full = O.evaluate(INJ[None], S, None, None, g, 1, o)
    Hd = O.dense_template(*INJ[[0, 1, 2, 7]], g, o)
    hh_m = (0.7 ** 2 + 0.5 ** 2) * np.sum(np.abs(Hd) ** 2, axis=1)
    assert abs(r["upsilon"][0] / full["upsilon"][0] - hh_m[gap != 0].sum() / hh_m.sum()) < 1e-10
    gap = np.ones(g.Nt, dtype=np.uint8); gap[128:256] = 0               # whole segment 1 of 4 masked
    r = O.evaluate(INJ[None], S + 0.0, None, gap, g, 4, o)
    assert r["seg_power"][0, 1] == 0.0 and r["seg_hh"][0, 1] == 0.0 and r["upsilon"][0] > 0


# ------------------------------------------------------------------------------------------
# P11 whole oracle vs a triple-loop re-implementation with a different Fresnel routine
# ------------------------------------------------------------------------------------------
def test_p11_triple_loop_reimplementation():
    mp = pytest.importorskip("mpmath")
    g = O.Grid(8, 32, 50.0)                                              # DT = 3200 s, df = 0.3125 mHz
    o = O.Opts(half_width=3)
    rng = np.random.default_rng(11)
    D = rng.standard_normal((2, 8, 32)) + 1j * rng.standard_normal((2, 8, 32))
    W = rng.uniform(0.5, 2, (2, 8, 32))
    gap = np.array([1, 1, 0, 1, 1, 1, 1, 1], dtype=np.uint8)
    # a (non-astrophysical) heavy system so that c = fdot DT^2 ~ 0.3-0.6 on this tiny grid and
    # the window is clipped at the upper band edge in the last tranches
    p = np.array([8000.0, 8.0e4, 0.9, 0.8, -0.1, 0.3, 0.4, 1.5])
    Nseg = 4
    res = O.evaluate(p[None], D, W, gap, g, Nseg, o)
    DT, df = 2 * g.Nf * g.dt, 1.0 / (2 * g.Nf * g.dt)
    M = p[0] * 4.925490947e-6
    T = [complex(p[3], p[4]), complex(p[5], p[6])]
    z = [0j] * Nseg
    hh = [0.0] * Nseg
    nact = 0
    for m in range(g.Nt):
        tau = p[1] - m * DT
        if gap[m] == 0 or tau <= DT:
            continue
        X = tau / (5 * M)
        f = X ** (-3.0 / 8.0) / (8 * math.pi * M)
        phi = p[2] - 2 * X ** (5.0 / 8.0)
        fdot = 3 * f / (8 * tau)
        if f < df or f + fdot * DT > (g.Nf - 1) * df or fdot * DT * DT > 300:
            continue
        nact += 1
        A = p[7] * f ** (2.0 / 3.0)
        kc = math.ceil(f / df)
        k_hi = math.ceil((f + fdot * DT) / df) + 3
        n = (m * Nseg) // g.Nt
        for k in range(max(kc - 3, 1), min(k_hi, g.Nf - 1) + 1):
            zeta = (f - k * df) / fdot                                   # Eq. 17
            v0 = math.sqrt(2 * fdot) * zeta                              # Eq. 22 at t_nm
            v1 = math.sqrt(2 * fdot) * (DT + zeta)                       # Eq. 22 at t_nm+1
            F = complex(mp.fresnelc(v1) - mp.fresnelc(v0), mp.fresnels(v1) - mp.fresnels(v0))
            h = A / math.sqrt(2 * fdot) * cmath.exp(1j * (phi - math.pi * fdot * zeta * zeta)) * F / DT
            for a in range(2):
                z[n] += T[a] * W[a, m, k] * D[a, m, k].conjugate() * h
                hh[n] += abs(T[a]) ** 2 * W[a, m, k] * abs(h) ** 2
    assert nact >= 5
    ups = sum(abs(zz) ** 2 / q for zz, q in zip(z, hh) if q > 0)
    assert np.allclose(res["seg_dh"][0], z, rtol=1e-9, atol=1e-12)
    assert np.allclose(res["seg_hh"][0], hh, rtol=1e-9)
    assert abs(res["upsilon"][0] / ups - 1) < 1e-9


# ------------------------------------------------------------------------------------------
# P12 truncation: N_F = 21 bins hold ~99 % of the power while the sweep is small
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("c,lo,hi", [(1e-4, 0.975, 0.995), (0.5, 0.975, 0.995), (3.0, 0.985, 0.999)])
def test_p12_window_power(c, lo, hi):
    fr = []
    for x in np.linspace(500.0, 501.0, 11, endpoint=False) + 0.013:
        k = np.arange(1, 1024)
        H = O.kernel_pixels(x, c, 0.0, 1.0, k)
        kc = math.ceil(x)
        win = (k >= kc - 10) & (k <= math.ceil(x + c) + 10)
        fr.append(np.sum(np.abs(H[win]) ** 2) / np.sum(np.abs(H) ** 2))
    assert lo < np.mean(fr) < hi


def test_p12_fixed_window_loses_fast_chirps():
    # DESIGN.md C4: the paper-strict 21 bins collapse once c >~ 10
    x, c = 500.3, 25.0
    k = np.arange(1, 1024)
    H = O.kernel_pixels(x, c, 0.0, 1.0, k)
    kc = math.ceil(x)
    fixed = (k >= kc - 10) & (k <= kc + 10)
    adapt = (k >= kc - 10) & (k <= math.ceil(x + c) + 10)
    tot = np.sum(np.abs(H) ** 2)
    assert np.sum(np.abs(H[fixed]) ** 2) / tot < 0.6
    assert np.sum(np.abs(H[adapt]) ** 2) / tot > 0.985


# ------------------------------------------------------------------------------------------
# track / window / segment bookkeeping
# ------------------------------------------------------------------------------------------
def test_track_closed_forms():
    g, o = TINY, O.Opts()
    tr = O.track(30.0, O.YEAR_S, 0.0, 1.0, g, o)
    # phase derivative: f = (1/2pi) dphi/dt (Eq. 14), fdot = df/dt (Eq. 15) by finite differences
    m = np.arange(1, g.Nt - 1)
    dphi = (tr["phi"][m + 1] - tr["phi"][m - 1]) / (2 * g.DT) / (2 * np.pi)
    assert np.max(np.abs(dphi / tr["f"][m] - 1)) < 1e-6
    dfdt = (tr["f"][m + 1] - tr["f"][m - 1]) / (2 * g.DT)
    assert np.max(np.abs(dfdt / tr["fdot"][m] - 1)) < 1e-5
    # the injection runs from 27.8 to 29.7 mHz
    assert abs(tr["f"][0] - 27.8e-3) < 1e-4 and abs(tr["f"][-1] - 29.7e-3) < 1e-4
    assert np.all(tr["k_hi"] - tr["k_lo"] + 1 >= 21) and np.all(tr["k_hi"] - tr["k_lo"] + 1 <= 22)
    # time to coalescence from f: tau = 5/256 M^{-5/3} (pi f)^{-8/3} (textbook 0PN)
    M = 30.0 * O.MTSUN_S
    tau = 5.0 / 256.0 * M ** (-5.0 / 3.0) * (np.pi * tr["f"][0]) ** (-8.0 / 3.0)
    assert abs(tau / O.YEAR_S - 1) < 1e-12


def test_inactive_and_bad_templates():
    g, o = SMALL, O.Opts()
    D = _noise(g, 3)
    P = np.array([[30.0, 100.0, 0, 1, 0, 0, 0, 1],           # tc <= DT: no active tranche
                  [5.0, 1e4, 0, 1, 0, 0, 0, 1],              # starts above the band
                  [np.nan, 1e7, 0, 1, 0, 0, 0, 1],
                  [30.0, np.inf, 0, 1, 0, 0, 0, 1]])
    r = O.evaluate(P, D, None, None, g, 4, o)
    assert np.all(r["upsilon"] == 0) and np.all(r["seg_hh"] == 0)


def test_segments_and_topk():
    assert list(O.segment_of_bin(np.arange(8), 8, 4)) == [0, 0, 1, 1, 2, 2, 3, 3]
    assert list(O.segment_of_bin(np.arange(7), 7, 3)) == [0, 0, 0, 1, 1, 2, 2]
    idx, val = O.topk(np.array([1.0, 5.0, 3.0, 5.0, 0.0]), 3)
    assert list(idx) == [1, 3, 2] and list(val) == [5.0, 5.0, 3.0]


# ------------------------------------------------------------------------------------------
# P13  ladder refinement lattice and ladder driver (BASELINE.json configs[4]; C19)
# ------------------------------------------------------------------------------------------
def test_p13_refine_offsets_written_out():
    # r = 4: the offsets the header prints, -3/8, -1/8, 1/8, 3/8 of the parent's cell
    p = np.array([[30.0, 1000.0, 0.1, 0.2, 0.3, 0.4, 0.5, 0.6], [7.0, 5.0e7, 1, 2, 3, 4, 5, 6]])
    ch = O.refine(p, [1, 0], 4, 1e-3, 800.0)
    assert ch.shape == (32, 8)
    offs = [-0.375, -0.125, 0.125, 0.375]
    for j, src in enumerate([1, 0]):
        for a in range(4):
            for b in range(4):
                row = ch[j * 16 + a * 4 + b]
                assert row[0] == p[src, 0] * (1.0 + offs[a] * 1e-3)
                assert row[1] == p[src, 1] + offs[b] * 800.0
                assert np.array_equal(row[2:], p[src, 2:])


@pytest.mark.parametrize("r", [1, 2, 3, 4, 5])
def test_p13_refine_tiles_the_parent_lattice(r):
    # parents on a regular tc lattice of step d: the children of all parents form ONE regular lattice
    # of step d/r (no hole, no overlap at cell borders); same in Mc to first order in d_mc_rel
    d_tc, d_mc = 640.0, 1e-4
    par = np.array([[50.0, 1e6 + i * d_tc, 0, 1, 0, 0, 0, 1] for i in range(5)])
    ch = O.refine(par, range(5), r, d_mc, d_tc)
    tcs = np.unique(ch[:, 1])
    assert len(tcs) == 5 * r
    assert np.allclose(np.diff(tcs), d_tc / r, rtol=0, atol=1e-6)
    assert abs(tcs.mean() - par[:, 1].mean()) < 1e-6          # children are centred on the parents
    parM = np.array([[50.0 * (1 + d_mc) ** i, 1e6, 0, 1, 0, 0, 0, 1] for i in range(5)])
    chM = O.refine(parM, range(5), r, d_mc, d_tc)
    lm = np.log(np.unique(chM[:, 0]))
    assert len(lm) == 5 * r
    assert np.allclose(np.diff(lm), d_mc / r, rtol=0, atol=2 * d_mc ** 2)
    # r = 1 is the identity
    if r == 1:
        assert np.array_equal(ch, par)


def test_p13_ladder_reduces_to_plain_evaluation():
    # keep everything, r = 1: every stage is O.evaluate of the same bank at that stage's N_seg
    g = SMALL
    D = _noise(g, 5)
    rng = np.random.default_rng(8)
    P = np.array([[rng.uniform(25, 35), rng.uniform(0.3, 3) * O.YEAR_S, 0.0, 0.6, 0.1, -0.3, 0.5, 1.0] for _ in range(6)])
    st = O.ladder(P, D, None, None, g, 1e-4, 100.0, stages=(8, 2, 1), keep_frac=1.0, r=1)
    for s, N in zip(st, (8, 2, 1)):
        u = O.evaluate(P, D, None, None, g, N)["upsilon"]
        assert np.array_equal(np.sort(s["upsilon"]), np.sort(u))
        assert list(s["top_idx"]) == list(O.topk(s["upsilon"], len(P))[0])


def test_p13_ladder_recovers_a_noiseless_injection():
    # a coarse lattice around (not on) the injection: each stage's survivors contain the cell that
    # holds the truth, the final candidate is within half a final step of it, and the recovered
    # coherent SNR^2 is most of rho^2 (hierarchical reduction of N_seg ends at the coherent limit)
    g = O.Grid(256, 1024, 5.0)
    inj = np.array([30.0, 1.0 * O.YEAR_S, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])
    S = O.injection(inj, 20.0, None, None, g)
    d_mc, d_tc, r = 4e-4, 2.0e4, 4
    nodes = np.arange(-3, 4)
    bank = []
    for i in nodes:
        for j in nodes:
            p = inj.copy()
            p[0] = inj[0] * (1.0 + (i + 0.31) * d_mc)
            p[1] = inj[1] + (j - 0.27) * d_tc
            p[2] = 0.0
            bank.append(p)
    bank = np.array(bank)
    st = O.ladder(bank, S, None, None, g, d_mc, d_tc, stages=(64, 16, 4, 1), keep_frac=0.05, r=r, keep_min=2)
    assert [len(s["params"]) for s in st] == [49, 48, 48, 48]
    # (Mc, tc) are degenerate along a ridge (a lighter system merging later has the same in-grid track),
    # so the best lattice point need not be in the truth's own cell; what the ladder must deliver is a
    # candidate near the truth in units of the FINAL step whose coherent SNR^2 is most of rho^2
    best = st[-1]["params"][st[-1]["top_idx"][0]]
    assert abs(best[0] / inj[0] - 1) <= 1.5 * st[-1]["d_mc_rel"]
    assert abs(best[1] - inj[1]) <= 1.5 * st[-1]["d_tc"]
    assert all(s["top_val"][0] > 0.9 * 400.0 for s in st)
    # without refinement the stage-0 lattice is far too coarse for the coherent statistic
    u1 = O.evaluate(bank, S, None, None, g, 1)["upsilon"]
    assert u1.max() < 0.5 * 400.0 < 0.9 * 400.0 < st[-1]["top_val"][0]


# ------------------------------------------------------------------------------------------
# P14 channels (1, 2, 3) and the per-tranche transfer factor T_alpha(f_nm) (Eq. 3, Eq. 7,
#     P:213 Eq. 29, "computed once per tranche for all frequency bins")
# ------------------------------------------------------------------------------------------
def test_p14_transfer_table_interpolation():
    tab = np.array([1 + 1j, 3 - 1j, 2 + 5j])
    f0, df = 0.01, 0.005
    # at the knots, half-way between them, and held outside
    f = np.array([0.01, 0.015, 0.02, 0.0125, 0.0175, 0.0, 0.5])
    want = np.array([tab[0], tab[1], tab[2], 0.5 * (tab[0] + tab[1]), 0.5 * (tab[1] + tab[2]), tab[0], tab[2]])
    assert np.allclose(O.transfer_at(tab, f0, df, f), want, rtol=0, atol=1e-14)
    # a table sampled from a straight line reproduces the line between its ends
    a, b = 0.3 - 0.2j, 40.0 + 10.0j
    knots = f0 + df * np.arange(7)
    f = np.linspace(knots[0], knots[-1], 1001)
    assert np.allclose(O.transfer_at(a + b * knots, f0, df, f), a + b * f, rtol=0, atol=1e-13)
    assert np.allclose(O.transfer_at(np.array([2 - 3j]), 0.0, 1.0, f), 2 - 3j)          # one knot: a constant


def _p14_data(C, seed=14):
    g = O.Grid(64, 128, 40.0)                                            # DT = 10240 s
    rng = np.random.default_rng(seed)
    D = rng.standard_normal((C, g.Nt, g.Nf)) + 1j * rng.standard_normal((C, g.Nt, g.Nf))
    W = rng.uniform(0.5, 2.0, (C, g.Nt, g.Nf))
    gap = np.ones(g.Nt, dtype=np.uint8)
    gap[20:24] = 0
    # heavy systems so that the track crosses a good part of the band of this small grid
    P = np.array([[1500.0, 1.2e6, 0.4, 0.6, -0.2, 0.3, 0.5, 1.2], [1500.0, 2.0e6, 1.9, -0.4, 0.1, 0.7, 0.2, 0.8]])
    return g, D, W, gap, P


def test_p14_constant_table_is_the_constant_factor():
    g, D, W, gap, P = _p14_data(2)
    ref = O.evaluate(P, D, W, gap, g, 4)
    tabs = np.stack([[[p[3] + 1j * p[4]], [p[5] + 1j * p[6]]] for p in P])            # [n][2][1]
    one = O.evaluate_tf(P, tabs, 0.0, 1.0, D, W, gap, g, 4)
    many = O.evaluate_tf(P, np.repeat(tabs, 5, axis=2), 1e-4, 2e-3, D, W, gap, g, 4)   # five equal knots
    for r in (one, many):
        assert np.allclose(r["seg_dh"], ref["seg_dh"], rtol=1e-12, atol=1e-12)
        assert np.allclose(r["seg_hh"], ref["seg_hh"], rtol=1e-12)
        assert np.allclose(r["upsilon"], ref["upsilon"], rtol=1e-12)


def test_p14_channel_counts():
    g, D, W, gap, P = _p14_data(3)
    two = O.evaluate(P, D[:2], W[:2], gap, g, 4)
    # a third channel without a transfer factor (T_T = 0) changes nothing, exactly
    three = O.evaluate(P, D, W, gap, g, 4)
    for k in ("upsilon", "seg_dh", "seg_hh"):
        assert np.array_equal(two[k], three[k])
    # ... and the same through a table whose third row is zero
    tabs = np.stack([[[p[3] + 1j * p[4]], [p[5] + 1j * p[6]], [0.0]] for p in P])
    t3 = O.evaluate_tf(P, tabs, 0.0, 1.0, D, W, gap, g, 4)
    assert np.allclose(t3["upsilon"], two["upsilon"], rtol=1e-12)
    # one channel = two channels with T_E = 0
    Q = P.copy()
    Q[:, 5:7] = 0.0
    one = O.evaluate(P, D[:1], W[:1], gap, g, 4)
    assert np.allclose(one["upsilon"], O.evaluate(Q, D[:2], W[:2], gap, g, 4)["upsilon"], rtol=1e-13)
    # three channels with three factors: the sum over alpha of Eq. 3, term by term
    tabs3 = np.stack([[[0.5 + 0.1j], [-0.2 + 0.6j], [0.3 - 0.3j]]] * len(P))
    full = O.evaluate_tf(P, tabs3, 0.0, 1.0, D, W, gap, g, 1)
    zsum, hsum = 0j, 0.0
    for a in range(3):
        ta = np.zeros((len(P), 1, 1), dtype=complex) + tabs3[:, a:a + 1]
        ra = O.evaluate_tf(P[:1], ta[:1], 0.0, 1.0, D[a:a + 1], W[a:a + 1], gap, g, 1)
        zsum += ra["seg_dh"][0, 0]
        hsum += ra["seg_hh"][0, 0]
    assert abs(full["seg_dh"][0, 0] - zsum) < 1e-10 * abs(zsum) and abs(full["seg_hh"][0, 0] - hsum) < 1e-12 * hsum


def test_p14_varying_transfer_noiseless_injection_and_loop():
    g, D, W, gap, P = _p14_data(3)
    p = P[0]
    f0, dfk, K = 7.5e-3, 0.6e-3, 6
    rng = np.random.default_rng(3)
    tab = rng.standard_normal((3, K)) + 1j * rng.standard_normal((3, K))
    tr = O.track(p[0], p[1], p[2], p[7], g, O.Opts(), gap)
    fa = tr["f"][tr["active"]]
    assert fa.min() < f0 + 2 * dfk and fa.max() > f0 + 5 * dfk            # the track crosses several knots and leaves the table
    # (i) noiseless injection carrying the same T_alpha(f_m): Upsilon_N = rho^2 for every N
    S = O.injection_tf(p, tab, f0, dfk, 17.0, W, gap, g, truncate=True)
    for N in (1, 4, 16):
        r = O.evaluate_tf(p[None], tab[None], f0, dfk, S, W, gap, g, N)
        assert abs(r["upsilon"][0] - 289.0) < 1e-8
    # ... while the factor frozen at its first-knot value loses power
    frozen = O.evaluate_tf(p[None], tab[None, :, :1], f0, dfk, S, W, gap, g, 1)
    assert frozen["upsilon"][0] < 0.9 * 289.0
    # (ii) the per-tranche factor against plain loops: z_n = sum_alpha sum_m T_alpha(f_m) sum_k W conj(D) H
    N = 4
    r = O.evaluate_tf(p[None], tab[None], f0, dfk, D, W, gap, g, N)
    Hd = O.dense_template(p[0], p[1], p[2], p[7], g, O.Opts(), gap)
    z = [0j] * N
    hh = [0.0] * N
    for m in range(g.Nt):
        if not tr["active"][m]:
            continue
        s = min(max((tr["f"][m] - f0) / dfk, 0.0), K - 1.0)
        j = min(int(math.floor(s)), K - 2)
        for a in range(3):
            T = tab[a, j] + (tab[a, j + 1] - tab[a, j]) * (s - j)
            n = (m * N) // g.Nt
            for k in range(int(tr["k_lo"][m]), int(tr["k_hi"][m]) + 1):
                z[n] += T * W[a, m, k] * np.conj(D[a, m, k]) * Hd[m, k]
                hh[n] += abs(T) ** 2 * W[a, m, k] * abs(Hd[m, k]) ** 2
    assert np.allclose(r["seg_dh"][0], z, rtol=1e-10, atol=1e-12) and np.allclose(r["seg_hh"][0], hh, rtol=1e-10)


# ----------------------------------------------------------------------------------------------
# P15  segments of fixed duration T_seg = M_tr DT ("t_n = n T_seg", P:57 N_seg = tau/T_seg, M_tr = T_seg/DT)
# ----------------------------------------------------------------------------------------------
def test_p15_fixed_duration_segments():
    rng = np.random.default_rng(15)
    g = O.Grid(48, 128, 5.0)
    D = rng.standard_normal((2, g.Nt, g.Nf)) + 1j * rng.standard_normal((2, g.Nt, g.Nf))
    W = rng.uniform(0.5, 2.0, (2, g.Nt, g.Nf))
    gap = (rng.uniform(size=g.Nt) > 0.2).astype(np.uint8)
    p = np.array([[30.0, 0.9 * g.Tobs, 0.3, 0.7, 0.1, 0.5, -0.2, 1.0],       # merges inside the grid
                  [22.0, 3.0 * g.Tobs, 1.0, 0.2, 0.0, 0.9, 0.3, 2.0]])
    # (a) M_tr divides Nt: the same numbers as the equal-index rule with N_seg = Nt / M_tr
    for M_tr in (1, 4, 12, 48):
        a = O.evaluate_tseg(p, D, W, gap, g, M_tr)
        b = O.evaluate(p, D, W, gap, g, g.Nt // M_tr)
        for k in ("upsilon", "seg_power", "seg_dh", "seg_hh"):
            assert np.array_equal(a[k], b[k]), (M_tr, k)
    # (b) ragged last segment, against plain loops over tranches: z_n, hh_n accumulated tranche by tranche
    M_tr = 10
    a = O.evaluate_tseg(p, D, W, gap, g, M_tr)
    assert a["seg_hh"].shape == (2, 5)
    for i in range(2):
        Hd = O.dense_template(p[i, 0], p[i, 1], p[i, 2], p[i, 7], g, O.Opts(), gap)
        T = [p[i, 3] + 1j * p[i, 4], p[i, 5] + 1j * p[i, 6]]
        z = np.zeros(5, dtype=complex); hh = np.zeros(5)
        for m in range(g.Nt):
            if not gap[m]:
                continue
            for al in range(2):
                z[m // M_tr] += T[al] * np.sum(W[al, m] * np.conj(D[al, m]) * Hd[m])
                hh[m // M_tr] += abs(T[al]) ** 2 * np.sum(W[al, m] * np.abs(Hd[m]) ** 2)
        assert np.allclose(a["seg_dh"][i], z, rtol=1e-12, atol=1e-12) and np.allclose(a["seg_hh"][i], hh, rtol=1e-12)
        assert a["n_seg_eff"][i] == int((hh > 0).sum())
    # (c) M_tr >= Nt: one segment, the coherent statistic
    assert np.array_equal(O.evaluate_tseg(p, D, W, gap, g, 1000)["upsilon"], O.evaluate(p, D, W, gap, g, 1)["upsilon"])


def test_p15_n_seg_eff_is_tau_over_tseg():
    """Without gaps and inside the band the number of occupied segments is ceil(tau / T_seg) with tau = min(T_obs, t_c - DT)
    rounded down to whole tranches: the paper's N_seg = tau / T_seg for tau = min(T_obs, t_c) on the tranche grid."""
    g = O.Grid(64, 512, 5.0)
    D = np.ones((1, g.Nt, g.Nf), dtype=complex)
    for frac in (0.13, 0.5, 0.77, 1.0, 4.0):
        tc = frac * g.Tobs
        p = np.array([[25.0, tc, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0]])
        n_active = int(min(g.Nt, math.ceil(tc / g.DT - 1.0)))         # tranches with tau = tc - m DT > DT
        o = O.Opts(f_lo=0.0, f_hi=1e9, c_max=1e300)                   # no band or sweep limit: only tau > DT cuts
        tr = O.track(25.0, tc, 0.0, 1.0, g, o)
        assert int(tr["active"].sum()) == n_active
        for M_tr in (1, 5, 16):
            r = O.evaluate_tseg(p, D, None, None, g, M_tr, o)
            assert r["n_seg_eff"][0] == math.ceil(n_active / M_tr), (frac, M_tr)


def test_p15_noise_mean_is_twice_n_seg_eff():
    """E[Upsilon] = 2 n_seg_eff for pure noise (each occupied segment contributes a chi^2_2), over 4000 noise draws of
    the window pixels of a template that merges inside the grid."""
    rng = np.random.default_rng(151)
    g = O.Grid(40, 256, 5.0)
    p = np.array([30.0, 0.62 * g.Tobs, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])
    M_tr = 6
    o = O.Opts(f_lo=0.0, f_hi=1e9, c_max=1e300)      # only the merger ends the track (its window is clipped to the top bin)
    Hd = O.dense_template(p[0], p[1], p[2], p[7], g, o)
    T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6]])
    seg = O.segment_of_bin_tseg(np.arange(g.Nt), M_tr)
    N_seg = -(-g.Nt // M_tr)
    ms, ks = np.nonzero(Hd)
    tot, n_draw = 0.0, 4000
    for _ in range(n_draw):
        D = np.zeros((2, g.Nt, g.Nf), dtype=complex)
        D[:, ms, ks] = rng.standard_normal((2, ms.size)) + 1j * rng.standard_normal((2, ms.size))
        z, hh = O.segment_products(Hd, T, D, None, None, N_seg, seg=seg)
        tot += O.combine(z, hh)[1]
    n_eff = int((hh > 0).sum())
    assert n_eff == math.ceil(int(O.track(p[0], p[1], 0, 1, g, o)["active"].sum()) / M_tr) and 1 < n_eff < N_seg
    mean, sig = tot / n_draw, 2.0 * math.sqrt(n_eff / n_draw)
    assert abs(mean - 2.0 * n_eff) < 4.0 * sig, (mean, n_eff)
