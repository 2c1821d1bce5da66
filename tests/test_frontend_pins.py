"""Pins of the front-end oracle (oracle/tfs_frontend.py)
against what the paper and the mathematics fix.  CPU only."""
import math

import numpy as np
import pytest

from oracle import tfs_frontend as F
from oracle import tfs_oracle as O


# F1  Tukey window ("Tukey-windowed with a shape parameter of 0.1")
@pytest.mark.parametrize("N,a", [(2048, 0.1), (6144, 0.1), (97, 0.1), (64, 0.5), (33, 1.0), (50, 0.0)])
def test_f1_tukey_window(N, a):
    from scipy.signal.windows import tukey as sp_tukey
    w = F.tukey(N, a)
    assert np.allclose(w, sp_tukey(N, a, sym=True), atol=1e-14)
    assert np.allclose(w, w[::-1], atol=1e-15) and w.max() <= 1.0 and w.min() >= 0.0
    if a == 0.0:
        assert (w == 1.0).all()
    else:
        assert w[0] == 0.0
        flat = (w == 1.0).mean()
        assert abs(flat - (1.0 - a)) < 2.5 / N + 1e-12          # a fraction 1 - a of the window is flat
    if a == 1.0:                                                  # Hann
        n = np.arange(N)
        assert np.allclose(w, 0.5 * (1 - np.cos(2 * np.pi * n / (N - 1))), atol=1e-14)


# F2  a tone that sits on a bin lands in that bin with amplitude A/2 and the tone's phase; DC -> mean(w)
@pytest.mark.parametrize("Nf", [64, 512])          # direct-sum path and FFT path of the oracle
def test_f2_tone_lands_in_its_bin(Nf):
    N, Nt, dt = 2 * Nf, 3, 5.0
    n = np.arange(Nt * N)
    k0, A, ph = 17, 2.5, 0.7
    x = np.stack([A * np.cos(2 * np.pi * k0 * n / N + ph), np.ones(Nt * N)])
    D, W, g = F.frontend(x, Nt, Nf, dt, tukey_alpha=0.0)
    expect = np.zeros(Nf, dtype=complex)
    expect[k0] = 0.5 * A * np.exp(1j * ph)
    assert np.allclose(D[0], expect[None, :], atol=1e-12)
    assert np.allclose(D[1][:, 0], 1.0, atol=1e-13) and np.allclose(D[1][:, 1:], 0.0, atol=1e-12)
    assert (W == 1.0).all() and (g == 1).all()
    Dw, _, _ = F.frontend(x, Nt, Nf, dt, tukey_alpha=0.1)
    assert np.allclose(Dw[1][:, 0], F.tukey(N, 0.1).mean(), atol=1e-13)


# F3  Parseval for the windowed tranche: sum (w x)^2 / N = |D_0|^2 + 2 sum_{0<k<Nf} |D_k|^2 + |D_Nyquist|^2
def test_f3_parseval():
    rng = np.random.default_rng(3)
    Nt, Nf, dt = 4, 384, 5.0
    N = 2 * Nf
    x = rng.standard_normal((2, Nt * N))
    D, _, _ = F.frontend(x, Nt, Nf, dt, tukey_alpha=0.1)
    w = F.tukey(N, 0.1)
    for a in range(2):
        for m in range(Nt):
            s = w * x[a, m * N:(m + 1) * N]
            nyq = (s * (-1.0) ** np.arange(N)).sum() / N
            lhs = (s * s).sum() / N
            rhs = abs(D[a, m, 0]) ** 2 + 2 * (np.abs(D[a, m, 1:]) ** 2).sum() + nyq ** 2
            assert abs(lhs - rhs) < 1e-12 * lhs


# F4  weights: white noise of one-sided PSD S = 2 sigma^2 dt gives E[W |D|^2] = 2 <w^2> in every interior bin
def test_f4_noise_weight_normalisation():
    rng = np.random.default_rng(4)
    Nt, Nf, dt, sigma = 400, 64, 5.0, 3.0
    N = 2 * Nf
    x = sigma * rng.standard_normal((1, Nt * N))
    S = np.full((1, Nf), 2 * sigma ** 2 * dt)
    D, W, _ = F.frontend(x, Nt, Nf, dt, psd=S, tukey_alpha=0.1)
    q = (W * np.abs(D) ** 2)[0][:, 1:]                      # [Nt][Nf-1], each ~ <w^2> chi^2_2
    w2 = (F.tukey(N, 0.1) ** 2).mean()
    mean, nsamp = q.mean(), q.size
    assert abs(mean - 2 * w2) < 4 * 2 * w2 / math.sqrt(nsamp)
    assert W.shape == (1, Nt, Nf) and np.allclose(W, 4 * N * dt / S[0, 0])
    # a PSD entry that is zero, negative or not finite gives weight 0
    S2 = S.copy(); S2[0, 0] = 0.0; S2[0, 5] = np.inf; S2[0, 6] = -1.0
    _, W2, _ = F.frontend(x[:, : 2 * N], 2, Nf, dt, psd=S2)
    assert (W2[0][:, [0, 5, 6]] == 0).all() and (W2[0][:, 1] > 0).all()


# F5  a tranche is valid iff all of its samples are
def test_f5_gap_mask():
    Nt, Nf = 6, 16
    N = 2 * Nf
    v = np.ones(Nt * N, dtype=np.uint8)
    v[N - 1] = 0                 # last sample of tranche 0
    v[3 * N] = 0                 # first sample of tranche 3
    v[4 * N + 5: 5 * N + 2] = 0  # a gap across tranches 4 and 5
    _, _, g = F.frontend(np.zeros((2, Nt * N)), Nt, Nf, 5.0, sample_mask=v)
    assert g.tolist() == [0, 1, 1, 0, 0, 0]


# F6  the front end feeds the hot path: a real 0PN chirp in the time domain, boxcar tranches, is recovered by the
#     template at the true parameters (BASELINE.json: within 2 % in SNR); with the paper's Tukey(0.1) window on the
#     data and the boxcar kernel of Eq. 16 as the template (the paper's own combination, C2) the loss
#     stays at the few-per-cent level of the windowed signal power
def test_f6_chirp_through_the_front_end():
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
    for alpha, lo in ((0.0, 0.98 ** 2), (0.1, 0.94)):
        D, W, gm = F.frontend(x, g.Nt, g.Nf, g.dt, tukey_alpha=alpha)
        w = F.tukey(N, alpha)
        rho2 = sum(((w[None, :] * x[a].reshape(g.Nt, N)) ** 2).sum() for a in range(2)) / (2 * N)
        r = O.evaluate(inj[None], D, None, gm, g, 1, O.Opts())
        assert lo < r["upsilon"][0] / rho2 < 1.0 + 1e-9, (alpha, r["upsilon"][0] / rho2)
