"""tfs_eval_tseg (segments of fixed duration T_seg = M_tr DT; per-template n_seg_eff) against the oracle
(O.evaluate_tseg).  n_seg_eff is integer work: exact.  Same bar as the other parity tests for the rest (C12)."""
import numpy as np
import pytest

from oracle import tfs_oracle as O
from paper_2510_19047_b200 import synth
from tests._common import assert_parity, to_complex

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


@pytest.mark.parametrize("Nt,Nf,weight_mode", [(333, 1024, 0), (150, 768, 1)])
def test_fixed_duration_segments_parity(api, Nt, Nf, weight_mode):
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=Nt, Nf=Nf, n_templates=60)
    coeff, weight, _ = synth.make_data(w)
    rng = np.random.default_rng(Nt)
    gap = (rng.uniform(size=Nt) > 0.15).astype(np.uint8)
    gap[40:75] = 0                                                           # and one whole segment of M_tr = 7 .. 16 missing
    params = synth.make_templates(w)
    params[:24, 0] = np.exp(rng.uniform(np.log(30.0), np.log(100.0), 24))
    params[:24, 1] = rng.uniform(0.05, 1.5, 24) * Nt * w.DT                 # merge inside or just after the grid
    params[3] = np.nan
    g = O.Grid(Nt, Nf, w.dt)
    D, W = to_complex(coeff), weight.astype(np.float64)
    ctx = api.Tfs(Nt, Nf, w.dt, weight_mode=weight_mode)
    ctx.upload_data(coeff, weight, gap)
    for M_tr in (1, 7, 64, 100, Nt, Nt + 5):
        gpu = api.eval_tseg_host(ctx, params, M_tr)
        ora = O.evaluate_tseg(params, D, W, gap, g, M_tr)
        N_seg = -(-Nt // M_tr)
        assert gpu["seg_hh"].shape == (len(params), N_seg)
        r = assert_parity(gpu, ora, N_seg, label=f"M_tr={M_tr}")
        assert r["n_active"] >= 25
        assert np.array_equal(gpu["n_seg_eff"], ora["n_seg_eff"]), M_tr          # integer: exact
        assert gpu["n_seg_eff"].max() > gpu["n_seg_eff"][gpu["n_seg_eff"] > 0].min() or N_seg == 1
    # M_tr | Nt == the equal-index rule of tfs_eval, bit for bit
    if Nt % 3 == 0:
        a = api.eval_tseg_host(ctx, params, Nt // 3)
        b = api.eval_host(ctx, params, 3)
        for k in ("upsilon", "seg_power", "seg_dh", "seg_hh"):
            assert np.array_equal(a[k], b[k]), k
    with pytest.raises(api.TfsError):
        api.eval_tseg_host(ctx, params, 0)
    ctx.destroy()


def test_tseg_device_buffers_and_nullable_outputs(api):
    import torch
    w = synth.scaled(synth.WORKLOADS["cfg2"], Nt=200, Nf=512, n_templates=500)
    coeff, weight, gap = synth.make_data(w)
    params = synth.make_templates(w)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    ctx.upload_data(coeff, weight, gap)
    ref = api.eval_tseg_host(ctx, params, 16)
    d_p = torch.from_numpy(params).cuda()
    d_u = torch.empty(len(params), dtype=torch.float32, device="cuda")
    d_n = torch.empty(len(params), dtype=torch.int32, device="cuda")
    ctx.eval_tseg(d_p, 16, d_u, d_n)
    torch.cuda.synchronize()
    assert np.array_equal(d_u.cpu().numpy(), ref["upsilon"]) and np.array_equal(d_n.cpu().numpy(), ref["n_seg_eff"])
    d_u.zero_()
    ctx.eval_tseg(d_p, 16, d_u)                                   # n_seg_eff omitted
    torch.cuda.synchronize()
    assert np.array_equal(d_u.cpu().numpy(), ref["upsilon"])
    ctx.destroy()
