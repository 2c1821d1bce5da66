"""Window-aware template (tfs_opts.tukey_alpha > 0; SURVEY.md 8(f) NEXT-2, P:271 vs P:153 Eq. 16, readings C2/C24)
on the GPU against the oracle (oracle/tfs_oracle.py: Opts.tukey_alpha).  Same bar as the other parity tests (C12)."""
import numpy as np
import pytest

from oracle import tfs_frontend as F
from oracle import tfs_oracle as O
from paper_2510_19047_b200 import synth
from tests._common import assert_parity, oracle_eval

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


def _bank(w, rng, fast_frac=0.4):
    """Templates as cfg2 plus a share that merges inside or just after the grid (c up to c_max, ragged windows)."""
    p = synth.make_templates(w)
    nf = int(fast_frac * len(p))
    p[:nf, 0] = np.exp(rng.uniform(np.log(30.0), np.log(100.0), nf))
    p[:nf, 1] = rng.uniform(0.05, 1.6, nf) * w.Nt * w.DT
    return p


@pytest.mark.parametrize("alpha,kind,Nt,Nf", [(0.1, "time", 200, 1024), (0.1, "general", 150, 768), (0.5, "product", 130, 1024),
                                              (1.0, "time", 70, 512), (0.02, "time", 90, 640)])
def test_windowed_template_parity(api, alpha, kind, Nt, Nf):
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=Nt, Nf=Nf, n_templates=64)
    rng = np.random.default_rng(int(alpha * 1000) + Nt)
    coeff = rng.standard_normal((2, Nt, Nf, 2)).astype(np.float32)
    a = rng.uniform(0.3, 2.0, (2, Nt, 1)).astype(np.float32)
    b = rng.uniform(0.5, 1.5, (2, 1, Nf)).astype(np.float32)
    weight = {"time": np.ascontiguousarray(np.broadcast_to(a, (2, Nt, Nf))), "product": (a * b).astype(np.float32),
              "general": rng.uniform(0.2, 3.0, (2, Nt, Nf)).astype(np.float32)}[kind]
    gap = (rng.uniform(size=Nt) > 0.12).astype(np.uint8)
    params = _bank(w, rng)
    ctx = api.Tfs(Nt, Nf, w.dt, tukey_alpha=alpha)
    ctx.upload_data(coeff, weight, gap)
    for N_seg in (1, 7, Nt):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = oracle_eval(coeff, weight, gap, params, Nt, Nf, w.dt, N_seg, tukey_alpha=alpha)
        r = assert_parity(gpu, ora, N_seg, label=f"alpha={alpha} {kind} N_seg={N_seg}")
        assert r["n_active"] >= 30
        # and the windowed result is NOT the boxcar one (the option does something)
        box = oracle_eval(coeff, weight, gap, params, Nt, Nf, w.dt, N_seg)
        act = ora["seg_hh"] > 0
        assert np.abs(ora["seg_hh"][act] / box["seg_hh"][act] - 1).max() > 5 * alpha * 0.1
    ctx.destroy()


def test_windowed_options(api):
    """Half widths 0 / 3 / 25, paper-strict window, wide tracks (c up to 300) with the window-aware template."""
    Nt, Nf = 96, 2048
    w = synth.scaled(synth.WORKLOADS["cfg4"], Nt=Nt, Nf=Nf, n_templates=48)
    rng = np.random.default_rng(5)
    coeff, weight, gap = synth.make_data(w)
    params = synth.make_templates(w)
    for opts in (dict(half_width=0), dict(half_width=3, adaptive_width=0), dict(half_width=25), dict(c_max=40.0)):
        ctx = api.Tfs(Nt, Nf, w.dt, tukey_alpha=0.1, **opts)
        ctx.upload_data(coeff, weight, gap)
        gpu = api.eval_host(ctx, params, 4)
        ora = oracle_eval(coeff, weight, gap, params, Nt, Nf, w.dt, 4, tukey_alpha=0.1, **opts)
        assert_parity(gpu, ora, 4, label=f"windowed {opts}")
        ctx.destroy()
    with pytest.raises(api.TfsError):
        api.Tfs(Nt, Nf, w.dt, tukey_alpha=1.5)
    with pytest.raises(api.TfsError):
        api.Tfs(Nt, Nf, w.dt, tukey_alpha=0.1, fresnel_mode=1)
    with pytest.raises(api.TfsError):
        api.Tfs(Nt, Nf, w.dt, tukey_alpha=0.1, basis=1)


def test_windowed_chirp_from_time_series(api):
    """End to end with the paper's combination done consistently: Tukey(0.1)-windowed tranches from
    tfs_upload_timeseries and the window-aware template.  Parity with the oracle chain, and the template at the
    true parameters recovers more of the windowed signal than the boxcar template does on the same data."""
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
    h *= 0.35 / np.abs(h).max()
    x = x + np.stack([((inj[3] + 1j * inj[4]) * h).real, ((inj[5] + 1j * inj[6]) * h).real]).astype(np.float32)
    params = np.vstack([synth.make_templates(w), inj[None]])
    Do, Wo, go = F.frontend(x, w.Nt, w.Nf, w.dt, sample_mask=mask, psd=psd, tukey_alpha=0.1)
    ups = {}
    for ta in (0.1, 0.0):
        ctx = api.Tfs(w.Nt, w.Nf, w.dt, tukey_alpha=ta)
        ctx.upload_timeseries(x, mask, psd, tukey_alpha=0.1)
        gpu = api.eval_host(ctx, params, 1)
        ora = O.evaluate(params, Do, Wo, go, g, 1, O.Opts(tukey_alpha=ta))
        assert_parity(gpu, ora, 1, label=f"time series, template alpha {ta}")
        ups[ta] = float(gpu["upsilon"][-1])
        ctx.destroy()
    assert ups[0.1] > 1.015 * ups[0.0] > 100.0, ups
