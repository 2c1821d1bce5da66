"""CPU oracle of the time-series -> time-frequency front end.

TEST INFRASTRUCTURE ONLY: imported by tests/ (and nothing else).  Plain numpy, fp64, no blocking or
reordering; shares no code with the CUDA path.

What it computes ("Each tranche is Tukey-windowed with a shape parameter of 0.1 and
fast-Fourier-transformed to construct the time-frequency grid"; "We model the noise PSD in each
tranche ..."; "tranches that overlap with data gaps are not included"):

  x[alpha, n]   real TDI time series, n = 0 ... Nt*N - 1, N = 2 Nf samples per tranche, cadence dt
  w[n]          Tukey window of length N with shape parameter a (fraction of the window inside the two cosine
                tapers): w[n] = (1 - cos(2 pi n / (a (N-1)))) / 2 for n < a (N-1)/2, mirrored at the other end,
                1 in between (Harris 1978; the symmetric form scipy.signal.windows.tukey implements)
  D[alpha,m,k]  = (1/N) sum_n w[n] x[alpha, m N + n] exp(-2 pi i k n / N),  k = 0 ... Nf-1
                (= dt * DFT / DT: the continuous-FT convention with the common factor DT dropped, as for the
                template kernel, C16)
  W[alpha,m,k]  = 4 DT / S_alpha[k]  for a one-sided PSD S [1/Hz] sampled at f_k = k/DT (0 where S is not
                positive and finite), so that E[W |D|^2] = 2 <w^2> for noise of that PSD; 1 when no PSD is given
  g[m]          = 1 iff every sample of tranche m is valid
"""
from __future__ import annotations

import numpy as np


def tukey(N: int, a: float) -> np.ndarray:
    """Symmetric Tukey (tapered cosine) window of length N, shape parameter a in [0, 1]."""
    if N == 1 or a <= 0.0:
        return np.ones(N)
    a = min(a, 1.0)
    n = np.arange(N, dtype=np.float64)
    edge = a * (N - 1) / 2.0
    w = np.ones(N)
    lo = n < edge
    hi = n > (N - 1) - edge
    w[lo] = 0.5 * (1.0 - np.cos(np.pi * n[lo] / edge))
    w[hi] = 0.5 * (1.0 - np.cos(np.pi * ((N - 1) - n[hi]) / edge))
    return w


def frontend(x, Nt: int, Nf: int, dt: float, sample_mask=None, psd=None, tukey_alpha: float = 0.1):
    """x [C][Nt*2*Nf] real -> (D [C][Nt][Nf] complex128, W [C][Nt][Nf] float64, g [Nt] uint8)."""
    x = np.asarray(x, dtype=np.float64)
    C = x.shape[0]
    N = 2 * Nf
    assert x.shape == (C, Nt * N)
    w = tukey(N, tukey_alpha)
    D = np.empty((C, Nt, Nf), dtype=np.complex128)
    n = np.arange(N)
    for a in range(C):
        for m in range(Nt):
            seg = w * x[a, m * N:(m + 1) * N]
            if N <= 256:            # small cases: the defining sum, written out
                k = np.arange(Nf)[:, None]
                D[a, m] = (seg[None, :] * np.exp(-2j * np.pi * k * n[None, :] / N)).sum(axis=1) / N
            else:                   # library primitive for the same sum
                D[a, m] = np.fft.fft(seg)[:Nf] / N
    DT = N * dt
    W = np.ones((C, Nt, Nf))
    if psd is not None:
        S = np.asarray(psd, dtype=np.float64)
        assert S.shape == (C, Nf)
        ok = np.isfinite(S) & (S > 0)
        Wk = np.where(ok, 4.0 * DT / np.where(ok, S, 1.0), 0.0)
        W = np.broadcast_to(Wk[:, None, :], (C, Nt, Nf)).copy()
    g = np.ones(Nt, dtype=np.uint8)
    if sample_mask is not None:
        v = np.asarray(sample_mask).reshape(Nt, N)
        g = (v != 0).all(axis=1).astype(np.uint8)
    return D, W, g
