"""Pins for the WDM-basis oracle (oracle/tfs_wdm.py) against what the mathematics fixes (SURVEY.md 8(f) NEXT-1:
"pin by Parseval only" -- ref. [28] is not in the container -- plus everything else that has a plain definition).
None of these call the CUDA path."""
import math

import numpy as np
import pytest

from oracle import tfs_oracle as O
from oracle import tfs_wdm as Wd


# W1-W3: the complete basis is orthonormal, for even and odd layer counts
@pytest.mark.parametrize("Nt,Nf", [(8, 8), (8, 7), (12, 6), (6, 5)])
def test_w_basis_is_orthonormal_and_complete(Nt, Nf):
    g = Wd.WdmGrid(Nt, Nf, 1.0)
    phi = Wd.window(g)
    assert abs(np.sum(phi ** 2) - 1.0) < 1e-13
    B = np.array([Wd.basis_function(n, m, g, phi) for n in range(Nt) for m in range(Nf)])
    assert B.shape == (g.N, g.N)
    assert np.abs(B @ B.T - np.eye(g.N)).max() < 1e-12                      # W^T W = I


def test_w_transform_reconstruction_parseval():
    g = Wd.WdmGrid(16, 12, 0.5)
    x = np.random.default_rng(5).standard_normal(g.N)
    wd = Wd.transform_direct(x, g)
    assert np.abs(Wd.transform(x, g) - wd).max() < 1e-12                    # FFT route == the sums written out
    assert np.abs(Wd.inverse_direct(wd, g) - x).max() < 1e-12
    assert abs(np.sum(wd ** 2) / np.sum(x ** 2) - 1.0) < 1e-12              # Parseval (BASELINE.json north_star)
    # white noise of unit variance gives unit-variance pixels
    big = Wd.WdmGrid(64, 64, 1.0)
    w = Wd.transform(np.random.default_rng(6).standard_normal(big.N), big)
    assert abs(np.var(w[:, 1:]) - 1.0) < 0.06


def test_w_stationary_tone_lands_in_two_adjacent_layers():
    g = Wd.WdmGrid(64, 32, 1.0)
    t = np.arange(g.N) * g.dt
    for xf in (5.0, 9.37, 17.5):                                            # tone frequency in layer units
        # (frequencies that fit the periodic series an integer number of times: no leakage from the wrap)
        f = round(xf * g.DF * g.N * g.dt) / (g.N * g.dt)
        w = Wd.transform(np.cos(2 * math.pi * f * t + 0.4), g)
        lay = np.sum(w ** 2, axis=0)
        m0 = int(math.floor(f / g.DF))
        assert lay[m0] + lay[min(m0 + 1, g.Nf - 1)] > (1 - 1e-12) * lay.sum()
        if abs(f / g.DF - round(f / g.DF)) < 1e-9:
            assert lay[m0] > (1 - 1e-12) * lay.sum()                        # on a layer centre: that layer alone


# W4: the chirp response
def test_w_response_limits_and_symmetry():
    x = np.linspace(-2.5, 2.5, 41)
    K0 = Wd.chirp_response(x, 0.0)
    assert np.allclose(K0, np.where(np.abs(x) < 1, np.cos(0.5 * math.pi * x), 0.0))
    Ks = Wd.chirp_response(x, 1e-4)                                         # slow chirp: the window's frequency response
    inside = np.abs(np.abs(x) - 1.0) > 0.1
    assert np.abs(Ks - K0)[inside].max() < 5e-3
    for kap in (0.05, 0.7, 3.0):
        K = Wd.chirp_response(x, kap)
        assert np.allclose(K, Wd.chirp_response(-x, kap), atol=1e-12)       # even window => even in x
    # Meyer condition: at kappa = 0 the two layers a tone sits between share its power exactly
    for off in (0.0, 0.3, 0.77):
        m = np.arange(-3, 4)
        assert abs(np.sum(np.abs(Wd.chirp_response(off - m, 0.0)) ** 2) - 1.0) < 1e-14


def test_w_response_closed_form_in_fresnel_integrals():
    """The closed form the oracle switches to for slow chirps (and the CUDA path evaluates) against the quadrature
    of the defining integral, on both sides of the switch, and its continuity across it."""
    x = np.linspace(-3, 3, 25)
    for kap in (1e-3, 0.01, 0.05, 0.5, 3.0):
        quad = Wd.chirp_response(x, max(kap, Wd.KAPPA_QUADRATURE_MIN)) if kap >= Wd.KAPPA_QUADRATURE_MIN else None
        if quad is None:
            # force the quadrature below the switch (slow: only here)
            saved = Wd.KAPPA_QUADRATURE_MIN
            Wd.KAPPA_QUADRATURE_MIN = 0.0
            try:
                quad = Wd.chirp_response(x, kap)
            finally:
                Wd.KAPPA_QUADRATURE_MIN = saved
        assert np.abs(Wd.chirp_response_closed(x, kap) - quad).max() < 1e-11
    k0 = Wd.KAPPA_QUADRATURE_MIN
    assert np.abs(Wd.chirp_response(x, k0 * (1 - 1e-9)) - Wd.chirp_response(x, k0)).max() < 1e-8


@pytest.mark.parametrize("kappa", [1e-3, 0.05, 0.5])
def test_w_template_pixel_is_the_transform_of_a_sampled_chirp(kappa):
    """Sign, phase, parity factor eps_nm and normalisation of W4: the exact WDM transform of a sampled linear chirp
    against A sqrt(Nf) Re[eps exp(i Phi_n) K] (sqrt(2 Nf) is the discrete window's peak response, dropped in W4)."""
    g = Wd.WdmGrid(64, 32, 1.0)
    t = np.arange(g.N) * g.dt
    fdot = kappa / (4 * g.DT ** 2)
    f0, Phi0, A = 9.3 * g.DF, 0.7, 1.3
    w = Wd.transform(A * np.cos(Phi0 + 2 * math.pi * f0 * t + math.pi * fdot * t * t), g)
    worst = 0.0
    for n in range(20, 44):
        tn = n * g.DT
        fn, Phin = f0 + fdot * tn, Phi0 + 2 * math.pi * f0 * tn + math.pi * fdot * tn * tn
        ms = np.arange(max(1, int(fn / g.DF) - 5), min(g.Nf - 1, int(fn / g.DF) + 6))
        H = Wd.eps(n, ms) * (A / math.sqrt(2)) * np.exp(1j * Phin) * Wd.chirp_response(fn / g.DF - ms, kappa)
        worst = max(worst, np.abs(math.sqrt(2 * g.Nf) * H.real - w[n, ms]).max())
    assert worst < 2.5e-3 * np.abs(w).max()


# W5-W7: the statistic
def _wdm_case(seed=3):
    g = Wd.WdmGrid(128, 64, 20.0)                                           # DT = 1280 s, DF = 0.39 mHz, 1.9 days
    rng = np.random.default_rng(seed)
    W = rng.uniform(0.5, 2.0, (2, g.Nt, g.Nf))
    gap = np.ones(g.Nt, dtype=np.uint8)
    gap[40:47] = 0
    p = np.array([2500.0, 3.2e5, 0.9, 0.6, -0.2, 0.3, 0.5, 1.1])           # heavy: sweeps ~10 layers on this small grid
    return g, W, gap, p


def test_w_noiseless_injection_gives_rho2_at_any_phase():
    g, W, gap, p = _wdm_case()
    tr = Wd.track(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(), gap)
    assert tr["active"].sum() > 80 and tr["xf"][tr["active"]].max() - tr["xf"][tr["active"]].min() > 5
    for phase in (0.0, 1.1, 2.7):
        S = Wd.injection(p, 13.0, W, gap, g, phase=phase)
        for N in (1, 4, 16):
            r = Wd.evaluate(p[None], S, W, gap, g, N)
            assert abs(r["upsilon"][0] - 169.0) < 1e-8                      # W6: maximised over amplitude AND phase
    # the two quadratures are nearly but not exactly orthogonal and equal (why W6 keeps the 2 x 2 Gram matrix)
    G = Wd.evaluate(p[None], S, W, gap, g, 1)["seg_gram"][0, 0]
    assert abs(G[0] / G[1] - 1) < 0.1 and abs(G[2]) < 0.1 * G[0] and (abs(G[0] / G[1] - 1) > 1e-6 or abs(G[2]) > 1e-6 * G[0])


def test_w_noise_only_expectation():
    g, W, gap, p = _wdm_case()
    H = Wd.dense_template(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(), gap)
    T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6]])
    rng = np.random.default_rng(12)
    for N in (1, 4, 16):
        ups = []
        for _ in range(1500):
            D = rng.standard_normal(W.shape) / np.sqrt(W)                    # E d^2 = 1/W
            z, G = Wd.segment_products(H, T, D, W, gap, N)
            ups.append(Wd.combine(z, G)[1])
        n_eff = int((Wd.segment_products(H, T, np.zeros_like(W), W, gap, N)[1][:, 0] > 0).sum())
        # each segment is maximised over two parameters: chi^2 with 2 degrees of freedom
        assert abs(np.mean(ups) - 2 * n_eff) < 3 * 2 * math.sqrt(n_eff / 1500.0)
        assert abs(np.var(ups) / (4 * n_eff) - 1) < 0.15


def test_w_layer_window_holds_the_power():
    g, W, gap, p = _wdm_case()
    Ht = Wd.dense_template(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(), gap, truncate=True)
    Hd = Wd.dense_template(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(), gap, truncate=False)
    assert np.sum(np.abs(Ht) ** 2) > 0.99 * np.sum(np.abs(Hd) ** 2)
    narrow = Wd.dense_template(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(half_width=0), gap, truncate=True)
    assert np.sum(np.abs(narrow) ** 2) < np.sum(np.abs(Ht) ** 2)


def test_w_time_domain_chirp_is_recovered():
    """A real 0PN chirp sampled in time, transformed exactly, is recovered by the method's template (W4: quadratic
    phase about the pixel centre, frozen amplitude) within BASELINE.json's 2 % in SNR."""
    g, W, gap, p = _wdm_case()
    t = np.arange(g.N) * g.dt
    M = p[0] * Wd.MTSUN_S
    tau = np.maximum(p[1] - t, 1e-3)
    X = tau / (5 * M)
    h = np.where(p[1] - t > 2.5 * g.DT, p[7] * (X ** (-0.375) / (8 * math.pi * M)) ** (2.0 / 3.0) * np.cos(p[2] - 2 * X ** 0.625), 0.0)
    wA = Wd.transform((p[3] * h), g)                                         # real antenna factors for this test
    wE = Wd.transform((p[5] * h), g)
    q = p.copy()
    q[4] = q[6] = 0.0
    D = np.stack([wA, wE])
    ones = np.ones_like(D)
    tr = Wd.track(q[0], q[1], q[2], q[7], g, Wd.WdmOpts(), None)
    act = tr["active"]
    rho2 = float(np.sum(D[:, act, 1:] ** 2))                                 # time-domain SNR^2 over the pixels the template uses
    r = Wd.evaluate(q[None], D, ones, None, g, 1)
    assert math.sqrt(r["upsilon"][0] / rho2) > 0.98


def _K_steepest_descent(x, kappa):
    """K(x, kappa) = e^{i pi/4}/sqrt(kappa) int_{-1}^{1} cos(pi y/2) exp(-i pi (y + x)^2/kappa) dy (W4's definition)
    by numerical steepest descent in mpmath: with w = y + x the integrand is entire, so the real segment is deformed
    into the paths of constant phase leaving each end point (w^2 = w_a^2 - i p, p >= 0, on which the exponential is
    exp(-i pi w_a^2/kappa) exp(-pi p/kappa)) plus, when the stationary point w = 0 lies between the end points, the
    straight line w = sqrt(kappa) e^{-i pi/4} s through it.  Every piece is a smooth decaying integral whatever kappa
    is; no Fresnel function and no completed square appear, so it shares nothing with the closed form it checks."""
    import mpmath as mp
    mp.mp.dps = 30
    x, kap = mp.mpf(x), mp.mpf(kappa)

    def endpoint(a):
        wa = a + x
        sg = 1 if wa > 0 else -1

        def f(q):                                                   # p = kappa q
            w = sg * mp.sqrt(wa * wa - 1j * kap * q)
            return mp.cos(mp.pi * (w - x) / 2) * mp.exp(-mp.pi * q) * (-1j * kap) / (2 * w)
        return mp.exp(-1j * mp.pi * wa * wa / kap) * mp.quad(f, [0, 1, 4, 16, mp.inf]), sg

    (Ilo, slo), (Ihi, shi) = endpoint(mp.mpf(-1)), endpoint(mp.mpf(1))
    tot = Ilo - Ihi
    if slo != shi:
        c = mp.sqrt(kap) * mp.exp(-0.25j * mp.pi)
        tot += mp.quad(lambda s: mp.cos(mp.pi * (c * s - x) / 2) * mp.exp(-mp.pi * s * s) * c, [-mp.inf, -2, 0, 2, mp.inf])
    return complex(tot * mp.exp(0.25j * mp.pi) / mp.sqrt(kap))


def test_w_response_closed_form_for_slow_chirps_by_steepest_descent():
    """Below kappa = 0.02 the oracle returns chirp_response_closed, the same Fresnel closed form the CUDA path
    evaluates, and the plain quadrature of the definition is only affordable down to kappa ~ 1e-3.  Slow chirps
    (c = 1e-4 ... 1e-3 give kappa = 4e-4 ... 4e-3, and the bank reaches 1e-6) are pinned here against an evaluation of
    the SAME defining integral that works at any kappa and uses neither Fresnel integrals nor the completed square.
    First the pin is itself checked against the Gauss-Legendre quadrature where that is cheap."""
    xs = [-2.3, -1.2, -0.999, -0.4, 0.013, 0.77, 1.0001, 1.9]          # inside, outside and at the edges of the window
    quad = Wd.chirp_response(np.array(xs), 0.5)
    assert np.abs(np.array([_K_steepest_descent(x, 0.5) for x in xs]) - quad).max() < 1e-12
    for kap in (4e-3, 1e-4, 1e-5, 1e-6):
        ref = np.array([_K_steepest_descent(x, kap) for x in xs])
        assert np.abs(Wd.chirp_response_closed(np.array(xs), kap) - ref).max() < 2e-12, kap
        assert np.array_equal(Wd.chirp_response(np.array(xs), kap), Wd.chirp_response_closed(np.array(xs), kap))
    # and the tone limit the oracle switches to below 1e-9 is what the integral tends to
    lim = Wd.chirp_response(np.array(xs), 1e-10)
    # (next to the window's edges |x| = 1 the end-point term is O(sqrt(kappa)) times the window's slope: 3e-6 at 1e-8)
    assert np.abs(np.array([_K_steepest_descent(x, 1e-8) for x in xs]) - lim).max() < 1e-5
