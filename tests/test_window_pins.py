"""Pins of the window-aware template kernel of the oracle (oracle/tfs_oracle.py: tukey_profile,
kernel_pixels_windowed_quad, kernel_pixels_windowed, reading C2/C24 of DESIGN.md).

The paper Tukey-windows every tranche before its FFT while Eq. 16 is the transform of the
un-windowed tranche; the window-aware kernel is Eq. 16's integrand times the window.  CPU only.
"""
import math

import numpy as np
import pytest

from oracle import tfs_oracle as O
from oracle import tfs_frontend as F


# WP1  the window profile: scipy's Tukey window sampled on the same points, end values, flat fraction
def test_wp1_profile_against_scipy():
    sig = pytest.importorskip("scipy.signal")
    for alpha in (0.0, 0.1, 0.35, 1.0):
        N = 4001
        s = np.arange(N) / (N - 1.0)                     # scipy's symmetric window samples s = n/(N-1)
        assert np.abs(O.tukey_profile(s, alpha) - sig.windows.tukey(N, alpha)).max() < 1e-12
    s = np.linspace(0, 1, 100001)
    w = O.tukey_profile(s, 0.1)
    assert w[0] == 0.0 and w[-1] == 0.0 and abs(w[2500] - 0.5) < 1e-12       # half height in the middle of the taper
    assert abs((w == 1.0).mean() - 0.9) < 1e-4                                 # a fraction 1 - alpha is flat


# WP2  alpha = 0 is Eq. 16: both the quadrature and the closed form reproduce kernel_pixels; alpha -> 0 continuously
def test_wp2_boxcar_limit():
    for c in (1e-4, 0.03, 2.0, 60.0):
        x = 700.37
        k = np.arange(688, 714 + int(c))
        ref = O.kernel_pixels(x, c, 0.4, 1.7, k)
        pk = np.abs(ref).max()
        assert np.abs(O.kernel_pixels_windowed_quad(x, c, 0.4, 1.7, k, 0.0) - ref).max() < 1e-10 * pk
        assert np.abs(O.kernel_pixels_windowed(x, c, 0.4, 1.7, k, 0.0) - ref).max() < 1e-10 * pk
        # a taper of length 1e-7 removes at most that fraction of the integral
        assert np.abs(O.kernel_pixels_windowed_quad(x, c, 0.4, 1.7, k, 2e-7) - ref).max() < 3e-7 * pk


# WP3  closed form (Fresnel integrals over the three stretches, cosines as frequency shifts) == the defining quadrature
def test_wp3_closed_form_against_quadrature():
    rng = np.random.default_rng(7)
    for alpha in (0.05, 0.1, 0.3, 0.77, 1.0):
        for c in (3e-5, 1e-3, 0.2, 1.0, 7.5, 33.0, 280.0):
            x = 500.0 + rng.uniform(-0.5, 0.5)
            k = np.arange(488, 514 + int(c))
            q = O.kernel_pixels_windowed_quad(x, c, 1.1, 0.9, k, alpha)
            f = O.kernel_pixels_windowed(x, c, 1.1, 0.9, k, alpha)
            assert np.abs(q - f).max() < 1e-9 * np.abs(q).max(), (alpha, c)


# WP4  c -> 0: the kernel is the Fourier transform of the window itself, A e^{i phi} int w(s) e^{2 pi i u s} ds,
#      written out here as a midpoint sum; and its value on the track (u = 0) is the window's mean 1 - alpha/2
def test_wp4_tone_limit_is_the_window_transform():
    alpha = 0.1
    Ns = 1 << 16
    s = (np.arange(Ns) + 0.5) / Ns
    w = 0.5 * (1 - np.cos(2 * np.pi * np.minimum(np.minimum(s, 1 - s), alpha / 2) / alpha))     # retyped, not imported
    x = 300.25
    k = np.arange(290, 312)
    ref = np.array([(w * np.exp(2j * np.pi * (x - kk) * s)).mean() for kk in k])
    # the defining quadrature at c = 1e-12 (no chirp left); the closed form at c = 1e-6, where the chirp still bends the
    # phase by pi c s^2 <= 3e-6 rad and the closed form's own phase pi u^2/c ~ 3e8 rad costs ~3e-8
    assert np.abs(O.kernel_pixels_windowed_quad(x, 1e-12, 0.0, 1.0, k, alpha) - ref).max() < 1e-9
    assert np.abs(O.kernel_pixels_windowed(x, 1e-6, 0.0, 1.0, k, alpha) - ref).max() < 3e-6
    on = O.kernel_pixels_windowed_quad(300.0, 1e-12, 0.0, 1.0, np.array([300]), alpha)[0]
    assert abs(on - (1 - alpha / 2)) < 1e-9


# WP5  against a sampled, windowed linear chirp Fourier-transformed numerically (the analogue of pin P2): the
#      front end's own convention D = (1/N) sum_n w[n] x[n] e^{-2 pi i k n / N} with scipy's sampled window
def test_wp5_sampled_windowed_chirp_fft():
    N = 8192
    n = np.arange(N)
    for alpha in (0.1, 0.5):
        w = F.tukey(N, alpha)
        for c in (1e-3, 0.4, 6.0, 45.0):
            x, phi, A = 1000.3, 0.9, 1.0
            s = n / N
            sig = A * np.exp(1j * (phi + 2 * np.pi * x * s + np.pi * c * s * s))
            D = np.fft.fft(w * sig) / N
            k = np.arange(985, 1016 + int(c))
            got = O.kernel_pixels_windowed(x, c, phi, A, k, alpha)
            box = O.kernel_pixels(x, c, phi, A, k)
            pk = np.abs(D[k]).max()
            assert np.abs(got - D[k]).max() < 3e-3 * pk, (alpha, c)
            assert np.abs(box - D[k]).max() > 2e-2 * pk          # the boxcar kernel of Eq. 16 is NOT what the FFT sees


# WP6  recovery through the front end (the analogue of F6): a real 0PN chirp, Tukey-windowed tranches; the
#      window-aware template recovers >= 0.99 of the windowed rho^2 where the boxcar template loses 2.5 % (a = 0.1)
#      and 17 % (a = 0.5)
def test_wp6_recovery_through_the_front_end():
    g = O.Grid(512, 1024, 5.0)
    inj = np.array([30.0, 1.0 * O.YEAR_S, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])
    N = 2 * g.Nf
    t = np.arange(g.Nt * N) * g.dt
    M = inj[0] * O.MTSUN_S
    X = (inj[1] - t) / (5 * M)
    f = X ** (-0.375) / (8 * np.pi * M)
    h = inj[7] * f ** (2.0 / 3.0) * np.exp(1j * (inj[2] - 2 * X ** 0.625))
    T = [inj[3] + 1j * inj[4], inj[5] + 1j * inj[6]]
    x = np.stack([(T[a] * h).real for a in range(2)])
    for alpha, box_hi in ((0.1, 0.98), (0.5, 0.85)):
        D, W, gm = F.frontend(x, g.Nt, g.Nf, g.dt, tukey_alpha=alpha)
        w = F.tukey(N, alpha)
        rho2 = sum(((w[None, :] * x[a].reshape(g.Nt, N)) ** 2).sum() for a in range(2)) / (2 * N)
        aware = O.evaluate(inj[None], D, None, gm, g, 1, O.Opts(tukey_alpha=alpha))["upsilon"][0] / rho2
        box = O.evaluate(inj[None], D, None, gm, g, 1, O.Opts())["upsilon"][0] / rho2
        assert 0.99 < aware < 1.0 + 1e-6, (alpha, aware)
        assert box < box_hi < aware, (alpha, box)


# WP7  noiseless injection with the windowed template: Upsilon_N = rho^2 for every N_seg (pin P5 for the new kernel)
def test_wp7_windowed_injection_rho2():
    g = O.Grid(64, 256, 5.0)
    o = O.Opts(tukey_alpha=0.1)
    p = np.array([28.0, 0.4 * O.YEAR_S, 1.0, 0.6, 0.2, -0.3, 0.5, 1.0])
    S = O.injection(p, 9.0, None, None, g, o, truncate=True)
    for N_seg in (1, 4, 16):
        r = O.evaluate(p[None], S, None, None, g, N_seg, o)
        assert abs(r["upsilon"][0] - 81.0) < 1e-8
