"""The statistic in the real-coefficient WDM wavelet pixel basis (tfs_opts.basis = 1) on the
GPU against oracle/tfs_wdm.py, element by element on the same seeded inputs, at the 1e-4 bar of the Fourier path
(normalised as DESIGN.md C12: z by max(|z|, sqrt(2 hh)), P by max(P, 2), Upsilon by max(Upsilon, 2 N_eff))."""
import numpy as np
import pytest

from oracle import tfs_wdm as Wd
from paper_2510_19047_b200 import synth

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


def _case(Nt, Nf, n, seed, C=2, heavy=False):
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=Nt, Nf=Nf, n_templates=n)
    g = Wd.WdmGrid(Nt, Nf, w.dt)
    rng = np.random.default_rng(seed)
    weight = rng.uniform(0.4, 2.5, (C, Nt, Nf)).astype(np.float32)
    coeff = (rng.standard_normal((C, Nt, Nf)) / np.sqrt(weight)).astype(np.float32)
    gap = (rng.uniform(size=Nt) > 0.12).astype(np.uint8)
    gap[Nt // 3: Nt // 3 + 9] = 0
    params = synth.make_templates(w)
    Tobs = Nt * g.DT
    params[: n // 2, 1] = rng.uniform(0.05, 3.0, n // 2) * Tobs             # many merge in or near the grid
    if heavy:
        params[:, 0] = np.exp(rng.uniform(np.log(30.0), np.log(3000.0), n))   # fast chirps: kappa up to the limit
        params[:, 1] = rng.uniform(0.2, 2.0, n) * Tobs
    return w, g, coeff, weight, gap, params


def _check(gpu, ora, N_seg, label):
    zo, ug, uo = ora["seg_dh"], gpu["upsilon"].astype(np.float64), ora["upsilon"]
    hh_o = 0.5 * (ora["seg_gram"][..., 0] + ora["seg_gram"][..., 1])
    hh_g = gpu["seg_hh"].astype(np.float64)
    n_eff = np.maximum((hh_o > 0).sum(axis=1), 1)
    e_hh = np.where(hh_o > 0, np.abs(hh_g - hh_o) / np.where(hh_o > 0, hh_o, 1.0), np.abs(hh_g))
    e_z = np.abs(gpu["seg_dh"] - zo) / np.maximum(np.maximum(np.abs(zo), np.sqrt(2.0 * hh_o)), 1e-300)
    e_z = np.where(hh_o > 0, e_z, np.abs(gpu["seg_dh"]))
    e_P = np.abs(gpu["seg_power"] - ora["seg_power"]) / np.maximum(ora["seg_power"], 2.0)
    e_u = np.abs(ug - uo) / np.maximum(uo, 2.0 * n_eff)
    r = dict(hh=e_hh.max(), z=e_z.max(), P=e_P.max(), ups=e_u.max(), n_active=int((uo > 0).sum()))
    assert max(r["hh"], r["z"], r["P"], r["ups"]) <= TOL, f"{label}: {r}"
    return r


@pytest.mark.parametrize("Nt,Nf,heavy", [(256, 512, False), (300, 384, True), (200, 640, False)])
def test_wdm_parity(api, Nt, Nf, heavy):
    w, g, coeff, weight, gap, params = _case(Nt, Nf, 64, 100 + Nt, heavy=heavy)
    # a signal to find: planted by the oracle at the parameters of the last row
    inj = np.array([40.0 if not heavy else 900.0, 1.6 * Nt * g.DT, 0.8, 0.5, 0.3, -0.4, 0.6, 1.0])
    coeff += Wd.injection(inj, 15.0, weight.astype(np.float64), gap, g, phase=0.7).astype(np.float32)
    params = np.vstack([params, inj[None]])
    ctx = api.Tfs(Nt, Nf, w.dt, 2, basis=1)
    ctx.upload_data(coeff, weight, gap)
    counts = np.empty(len(params), dtype=np.int64)
    ctx.count_pixels(params, counts)
    ref = []
    for p in params:
        tr = Wd.track(p[0], p[1], p[2], p[7], g, Wd.WdmOpts(), gap)
        ref.append(int((tr["m_hi"] - tr["m_lo"] + 1)[tr["active"]].sum()))
    assert np.array_equal(counts, np.array(ref))
    kmax = max(Wd.track(p[0], p[1], 0, 1, g, Wd.WdmOpts(), gap)["kappa"][Wd.track(p[0], p[1], 0, 1, g, Wd.WdmOpts(), gap)["active"]].max(initial=0.0)
               for p in params)
    assert kmax > (1.0 if heavy else 1e-4)
    for N_seg in (1, 7, 32):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = Wd.evaluate(params, coeff.astype(np.float64), weight.astype(np.float64), gap, g, N_seg)
        r = _check(gpu, ora, N_seg, f"wdm {Nt}x{Nf} heavy={heavy} N_seg={N_seg}")
        assert r["n_active"] >= 30
        # the injection stands out at its own parameters (non-central chi^2)
        assert abs(gpu["upsilon"][-1] - (225.0 + 2 * N_seg)) < 5 * np.sqrt(4 * N_seg + 4 * 225.0)
    ctx.destroy()


def test_wdm_single_channel_options_and_errors(api):
    w, g, coeff, weight, gap, params = _case(160, 256, 40, 7, C=1)
    ctx = api.Tfs(160, 256, w.dt, 1, basis=1, wdm_half_width=4, wdm_kappa_max=2.0)
    ctx.upload_data(coeff, weight, gap)
    gpu = api.eval_host(ctx, params, 5)
    ora = Wd.evaluate(params, coeff.astype(np.float64), weight.astype(np.float64), gap, g, 5,
                      Wd.WdmOpts(half_width=4, kappa_max=2.0))
    _check(gpu, ora, 5, "wdm C=1 Hw=4")
    with pytest.raises(api.TfsError):
        api.Tfs(160, 256, w.dt, 3, basis=1)                                  # one or two channels in this basis
    with pytest.raises(api.TfsError):
        ctx.eval_tf(params, 5, np.zeros((len(params), 1, 1, 2), dtype=np.float32), 1, 0.0, 1.0,
                    np.empty(len(params), dtype=np.float32))
    ctx.destroy()
