"""GPU parity of the time-series front end (tfs_upload_timeseries) against
oracle/tfs_frontend.py, element by element, and end to end through tfs_eval."""
import numpy as np
import pytest

from oracle import tfs_frontend as F
from oracle import tfs_oracle as O
from paper_2510_19047_b200 import synth
from tests._common import assert_parity

pytestmark = pytest.mark.gpu

# fp32 shared-memory FFT against the fp64 oracle: rounding ~ eps * log2(N) of the tranche's largest coefficient
TOL_D = 1e-6          # measured 1.0e-7 ... 1.3e-7


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need cuda:0 (libtfs has no CPU fallback)"
    from paper_2510_19047_b200 import api as _api
    _api.load_library()
    return _api


def _run(api, w, x, mask, psd, alpha, device=False):
    import torch
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    npix = 2 * w.Nt * w.Nf
    if device:
        dev = torch.device("cuda:0")
        tx, tm, tp = torch.from_numpy(x).to(dev), torch.from_numpy(mask).to(dev), torch.from_numpy(psd).to(dev)
        tc = torch.empty(2 * npix, dtype=torch.float32, device=dev)
        tw = torch.empty(npix, dtype=torch.float32, device=dev)
        tg = torch.empty(w.Nt, dtype=torch.uint8, device=dev)
        ctx.upload_timeseries(tx, tm, tp, alpha, tc, tw, tg)
        torch.cuda.synchronize()
        c, wt, g = tc.cpu().numpy(), tw.cpu().numpy(), tg.cpu().numpy()
    else:
        c = np.empty(2 * npix, dtype=np.float32)
        wt = np.empty(npix, dtype=np.float32)
        g = np.empty(w.Nt, dtype=np.uint8)
        ctx.upload_timeseries(x, mask, psd, alpha, c, wt, g)
    c = c.reshape(2, w.Nt, w.Nf, 2)
    return ctx, c[..., 0].astype(np.float64) + 1j * c[..., 1], wt.reshape(2, w.Nt, w.Nf), g


@pytest.mark.parametrize("Nf,Nt,alpha", [(1024, 12, 0.1), (3072, 6, 0.1), (768, 9, 0.0), (640, 7, 0.5), (1500, 5, 0.1),
                                         (2, 40, 0.1), (96, 33, 1.0)])
def test_frontend_parity(api, Nf, Nt, alpha):
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=Nt, Nf=Nf)
    x, mask, psd = synth.make_timeseries(w)
    ctx, D, W, g = _run(api, w, x, mask, psd, alpha, device=(Nf == 1024))
    Do, Wo, go = F.frontend(x, w.Nt, w.Nf, w.dt, sample_mask=mask, psd=psd, tukey_alpha=alpha)
    assert np.array_equal(g, go)                                           # byte work: exact
    scale = np.abs(Do).max(axis=2, keepdims=True)
    assert (np.abs(D - Do) <= TOL_D * scale).all(), float((np.abs(D - Do) / scale).max())
    assert np.allclose(W, Wo, rtol=3e-7, atol=0.0)                         # one fp32 division
    assert ctx.weight_structure() == (1 if Nf > 2 else ctx.weight_structure())
    ctx.destroy()


def test_frontend_rejects_unsupported_lengths(api):
    w = synth.scaled(synth.WORKLOADS["cfg1"], Nt=4, Nf=7 * 64)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    with pytest.raises(api.TfsError):
        ctx.upload_timeseries(np.zeros((2, w.Nt * 2 * w.Nf), dtype=np.float32))
    with pytest.raises(api.TfsError):
        api.Tfs(4, 64, 5.0).upload_timeseries(np.zeros((2, 4 * 128), dtype=np.float32), tukey_alpha=1.5)
    ctx.destroy()


def test_chirp_from_time_series_to_upsilon(api):
    """End to end: a real 0PN chirp plus noise in the time domain -> tfs_upload_timeseries -> tfs_eval, against
    the oracle front end followed by the oracle statistic, on the same series."""
    w = synth.scaled(synth.WORKLOADS["cfg1"], Nt=256, Nf=1024, n_templates=40)
    x, mask, psd = synth.make_timeseries(w)
    g = O.Grid(w.Nt, w.Nf, w.dt)
    inj = np.array([30.0, 1.0 * O.YEAR_S, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])
    N = 2 * w.Nf
    t = np.arange(w.Nt * N) * w.dt
    M = inj[0] * O.MTSUN_S
    X = (inj[1] - t) / (5 * M)
    f = X ** (-0.375) / (8 * np.pi * M)
    h = f ** (2.0 / 3.0) * np.exp(1j * (inj[2] - 2 * X ** 0.625))
    h *= 0.35 / np.abs(h).max()                                            # a loud chirp under unit-variance noise
    x = x + np.stack([((inj[3] + 1j * inj[4]) * h).real, ((inj[5] + 1j * inj[6]) * h).real]).astype(np.float32)
    params = np.vstack([synth.make_templates(w), inj[None]])
    ctx, D, W, gm = _run(api, w, x, mask, psd, 0.1)
    Do, Wo, go = F.frontend(x, w.Nt, w.Nf, w.dt, sample_mask=mask, psd=psd, tukey_alpha=0.1)
    for N_seg in (1, 8):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = O.evaluate(params, Do, Wo, go, g, N_seg, O.Opts())
        r = assert_parity(gpu, ora, N_seg, label=f"time series N_seg={N_seg}")
        assert r["n_active"] >= 30
    assert np.argmax(gpu["upsilon"]) == len(params) - 1 and gpu["upsilon"][-1] > 100.0
    ctx.destroy()


def test_two_tranche_lengths_from_one_series(api):
    """tranches of 6 h for f_in below 10 mHz and 3 h above.  One context has one tranche length, so the split is
    two contexts over the same series, (Nt, Nf) and (2 Nt, Nf/2); each runs through tfs_upload_timeseries + tfs_eval
    against the oracle chain, and the fast high-band chirp is recovered at least as well by the short tranches."""
    Nt, Nf = 96, 2048                                  # DT = 20480 s (5.7 h) and 10240 s (2.8 h) at dt = 5 s
    w = synth.scaled(synth.WORKLOADS["cfg1"], Nt=Nt, Nf=Nf, n_templates=16)
    x, mask, psd = synth.make_timeseries(w)
    inj = np.array([60.0, 0.35 * O.YEAR_S, 0.3, 0.7, 0.0, 0.5, 0.0, 1.0])          # f ~ 27 -> 40 mHz: the high band
    N = 2 * Nf
    t = np.arange(Nt * N) * w.dt
    M = inj[0] * O.MTSUN_S
    X = (inj[1] - t) / (5 * M)
    f = X ** (-0.375) / (8 * np.pi * M)
    h = f ** (2.0 / 3.0) * np.exp(1j * (inj[2] - 2 * X ** 0.625))
    h *= 0.35 / np.abs(h).max()
    x = x + np.stack([((inj[3] + 1j * inj[4]) * h).real, ((inj[5] + 1j * inj[6]) * h).real]).astype(np.float32)
    params = np.vstack([synth.make_templates(w), inj[None]])
    ups = {}
    for nt, nf in ((Nt, Nf), (2 * Nt, Nf // 2)):
        g = O.Grid(nt, nf, w.dt)
        psd_b = np.ascontiguousarray(psd[:, :: Nf // nf])                           # the same PSD model on the coarser bins
        ctx = api.Tfs(nt, nf, w.dt)
        ctx.upload_timeseries(x, mask, psd_b, tukey_alpha=0.0)
        gpu = api.eval_host(ctx, params, 1)
        Do, Wo, go = F.frontend(x, nt, nf, w.dt, sample_mask=mask, psd=psd_b, tukey_alpha=0.0)
        ora = O.evaluate(params, Do, Wo, go, g, 1, O.Opts())
        assert_parity(gpu, ora, 1, label=f"tranches of {2 * nf * w.dt:.0f} s")
        ups[nt] = float(gpu["upsilon"][-1])
        ctx.destroy()
    assert ups[2 * Nt] > 0.98 * ups[Nt] > 50.0, ups


def test_non_finite_samples_drop_their_tranche(api):
    """C20 for the front end: a NaN or Inf sample makes its tranche a gap (in any channel); everything else is unchanged."""
    w = synth.scaled(synth.WORKLOADS["cfg1"], Nt=24, Nf=256, n_templates=12)
    x, mask, psd = synth.make_timeseries(w)
    N = 2 * w.Nf
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    g0 = np.empty(w.Nt, dtype=np.uint8)
    ctx.upload_timeseries(x, mask, psd, tukey_alpha=0.1, gap_out=g0)
    ref = api.eval_host(ctx, synth.make_templates(w), 2)
    good = np.nonzero(g0)[0]
    xb = x.copy()
    xb[0, good[1] * N + 7] = np.nan
    xb[1, good[3] * N + N - 1] = np.inf
    g1 = np.empty(w.Nt, dtype=np.uint8)
    ctx.upload_timeseries(xb, mask, psd, tukey_alpha=0.1, gap_out=g1)
    want = g0.copy(); want[[good[1], good[3]]] = 0
    assert np.array_equal(g1, want)
    r = api.eval_host(ctx, synth.make_templates(w), 2)
    assert all(np.isfinite(r[k]).all() for k in ("upsilon", "seg_power", "seg_hh"))
    # the same result as masking those two tranches by hand
    m2 = mask.copy(); m2[good[1] * N] = 0; m2[good[3] * N] = 0
    ctx.upload_timeseries(x, m2, psd, tukey_alpha=0.1)
    r2 = api.eval_host(ctx, synth.make_templates(w), 2)
    assert np.array_equal(r["upsilon"], r2["upsilon"]) and not np.array_equal(r["upsilon"], ref["upsilon"])
    ctx.destroy()


def test_time_series_upload_with_paper_fresnel_mode(api):
    """fresnel_mode = 1 always evaluates with the per-pixel-weight kernel, so tfs_upload_timeseries must materialise W
    even with weight_mode = 0 and no weight_out (it once took the per-bin-table shortcut and left W unwritten).  A first
    upload with different weights on the same context makes stale weights visible if the second upload skips W.
    Tolerance 2e-3 as in test_paper_fresnel_mode (the printed approximants' branch discontinuity, reading C8)."""
    w = synth.scaled(synth.WORKLOADS["cfg1"], Nt=64, Nf=512, n_templates=24)
    x, mask, psd = synth.make_timeseries(w)
    g = O.Grid(w.Nt, w.Nf, w.dt)
    params = synth.make_templates(w)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, fresnel_mode=1)
    ctx.upload_timeseries(x, mask, np.ascontiguousarray(psd * 7.0), tukey_alpha=0.1)      # stale weights: 1/7 of the right ones
    ctx.upload_timeseries(x, mask, psd, tukey_alpha=0.1)
    Do, Wo, go = F.frontend(x, w.Nt, w.Nf, w.dt, sample_mask=mask, psd=psd, tukey_alpha=0.1)
    for N_seg in (1, 4):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = O.evaluate(params, Do, Wo, go, g, N_seg, O.Opts(fresnel_mode=1))
        r = assert_parity(gpu, ora, N_seg, tol=2e-3, label=f"time series, fresnel_mode=1, N_seg={N_seg}")
        assert r["n_active"] >= 12
    ctx.destroy()
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, fresnel_mode=1)                                       # and without a PSD: W = 1
    ctx.upload_timeseries(x, mask, None, tukey_alpha=0.0)
    Do, Wo, go = F.frontend(x, w.Nt, w.Nf, w.dt, sample_mask=mask, psd=None, tukey_alpha=0.0)
    gpu = api.eval_host(ctx, params, 2)
    ora = O.evaluate(params, Do, Wo, go, g, 2, O.Opts(fresnel_mode=1))
    assert_parity(gpu, ora, 2, tol=2e-3, label="time series, fresnel_mode=1, no PSD")
    ctx.destroy()
