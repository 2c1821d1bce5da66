"""Channels (1, 2, 3) and the per-tranche transfer factor T_alpha(f_nm) of tfs_eval_tf against the oracle
(Eq. 3, Eq. 7, Eq. 29).  Same bar as the other parity tests (C12)."""
import numpy as np
import pytest

from oracle import tfs_oracle as O
from paper_2510_19047_b200 import synth
from tests._common import TOL, assert_parity, to_complex

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


def _data(C, Nt=300, Nf=1024, n=72, seed=31, kind="time"):
    """C-channel noise with per-channel weights, gaps, and a bank with ragged tracks."""
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=Nt, Nf=Nf, n_templates=n)
    rng = np.random.default_rng(seed)
    coeff = rng.standard_normal((C, Nt, Nf, 2)).astype(np.float32)
    a = rng.uniform(0.3, 2.0, (C, Nt, 1)).astype(np.float32)
    b = rng.uniform(0.5, 1.5, (C, 1, Nf)).astype(np.float32)
    if kind == "time":
        weight = np.ascontiguousarray(np.broadcast_to(a, (C, Nt, Nf)))
    elif kind == "product":
        weight = (a * b).astype(np.float32)
    else:
        weight = rng.uniform(0.2, 3.0, (C, Nt, Nf)).astype(np.float32)
    gap = (rng.uniform(size=Nt) > 0.15).astype(np.uint8)
    params = synth.make_templates(w)
    params[: n // 2, 1] = rng.uniform(0.0, 3.0, n // 2) * Nt * w.DT
    return w, coeff, weight, gap, params


def _oracle(params, coeff, weight, gap, w, N_seg, tables=None, f0=0.0, dfk=1.0):
    g = O.Grid(w.Nt, w.Nf, w.dt)
    D, W = to_complex(coeff), weight.astype(np.float64)
    if tables is None:
        return O.evaluate(params, D, W, gap, g, N_seg)
    return O.evaluate_tf(params, tables[..., 0] + 1j * tables[..., 1], f0, dfk, D, W, gap, g, N_seg)


@pytest.mark.parametrize("C,kind", [(1, "time"), (1, "general"), (3, "product"), (2, "product")])
def test_constant_factors_per_channel_count(api, C, kind):
    w, coeff, weight, gap, params = _data(C, kind=kind)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, C)
    ctx.upload_data(coeff, weight, gap)
    assert ctx.weight_structure() == {"time": 2, "product": 1, "general": 0}[kind]
    if C == 3:
        # the row has no column for T_T: tfs_eval refuses until the caller states it (never a silent 2-channel statistic)
        with pytest.raises(api.TfsError) as e:
            api.eval_host(ctx, params, 1)
        assert e.value.code == api.TFS_EINVAL and "tfs_set_third_channel_factor" in str(e.value)
        ctx.set_third_channel_factor(0.0, 0.0)                         # channel T left out on purpose
    for N_seg in (1, 9):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = _oracle(params, coeff, weight, gap, w, N_seg)            # three channels: T_T = 0
        r = assert_parity(gpu, ora, N_seg, label=f"C={C} {kind} N_seg={N_seg}")
        assert r["n_active"] >= 30
    ctx.destroy()


@pytest.mark.parametrize("kind", ["time", "product", "general"])
def test_third_channel_constant_factor(api, kind):
    """A, E, T with constant factors (Eq. 3): T_A, T_E from the row, T_T from tfs_set_third_channel_factor,
    against the oracle's evaluate_tf with one-knot tables holding the same three constants; tfs_eval_tseg takes the
    same constant; a table passed to tfs_eval_tf overrides it."""
    w, coeff, weight, gap, params = _data(3, kind=kind, seed=77)
    n = len(params)
    t3 = 0.4 - 0.7j
    tables = np.empty((n, 3, 1, 2))
    tables[:, 0, 0, 0], tables[:, 0, 0, 1] = params[:, 3], params[:, 4]
    tables[:, 1, 0, 0], tables[:, 1, 0, 1] = params[:, 5], params[:, 6]
    tables[:, 2, 0, 0], tables[:, 2, 0, 1] = t3.real, t3.imag
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, 3)
    ctx.upload_data(coeff, weight, gap)
    ctx.set_third_channel_factor(t3.real, t3.imag)
    two = _oracle(params, coeff, weight, gap, w, 1)["upsilon"]
    for N_seg in (1, 6):
        gpu = api.eval_host(ctx, params, N_seg)
        ora = _oracle(params, coeff, weight, gap, w, N_seg, tables, 0.0, 1.0)
        r = assert_parity(gpu, ora, N_seg, label=f"A,E,T constant {kind} N_seg={N_seg}")
        assert r["n_active"] >= 30
    assert np.max(np.abs(_oracle(params, coeff, weight, gap, w, 1, tables, 0.0, 1.0)["upsilon"] - two)) > 0.1   # T matters
    # fixed-duration segments: Nt = 300, 50 tranches per segment == N_seg = 6 (the equal-index rule, P15)
    ts = api.eval_tseg_host(ctx, params, 50)
    assert_parity(ts, ora, 6, label=f"A,E,T constant {kind} tseg")
    # a table overrides the constant
    tab2 = np.random.default_rng(5).standard_normal((n, 3, 3, 2)).astype(np.float32)
    gpu = api.eval_host(ctx, params, 6, transfer=tab2, f_knot0=4e-3, f_knot_step=0.03)
    ora2 = _oracle(params, coeff, weight, gap, w, 6, tab2.astype(np.float64), 4e-3, 0.03)
    assert_parity(gpu, ora2, 6, label=f"A,E,T table over constant {kind}")
    with pytest.raises(api.TfsError):
        api.Tfs(w.Nt, w.Nf, w.dt, 2).set_third_channel_factor(1.0, 0.0)
    ctx.destroy()


@pytest.mark.parametrize("C,K,kind", [(2, 1, "time"), (2, 7, "time"), (3, 1, "time"), (3, 5, "product"), (3, 6, "general"),
                                      (1, 4, "product")])
def test_transfer_tables(api, C, K, kind):
    w, coeff, weight, gap, params = _data(C, kind=kind, seed=40 + C + K)
    n = len(params)
    rng = np.random.default_rng(7)
    tables = rng.standard_normal((n, C, K, 2)).astype(np.float32)
    # knots across the band the bank's tracks cross (the table is held constant outside them)
    f0, dfk = 4e-3, 0.06 / max(K - 1, 1)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, C)
    ctx.upload_data(coeff, weight, gap)
    for N_seg in (1, 6):
        gpu = api.eval_host(ctx, params, N_seg, transfer=tables, f_knot0=f0, f_knot_step=dfk)
        ora = _oracle(params, coeff, weight, gap, w, N_seg, tables.astype(np.float64), f0, dfk)
        r = assert_parity(gpu, ora, N_seg, label=f"C={C} K={K} {kind} N_seg={N_seg}")
        assert r["n_active"] >= 30
    if K > 1:
        # the table matters: freezing it at its first knot gives different numbers
        frozen = api.eval_host(ctx, params, 1, transfer=np.ascontiguousarray(tables[:, :, :1]), f_knot0=f0, f_knot_step=dfk)
        assert np.max(np.abs(frozen["upsilon"] - gpu["upsilon"])) > 0.1
    ctx.destroy()


def test_transfer_table_device_pointers_and_errors(api):
    import torch
    w, coeff, weight, gap, params = _data(3, n=40)
    n = len(params)
    tables = np.random.default_rng(1).standard_normal((n, 3, 4, 2)).astype(np.float32)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt, 3)
    ctx.upload_data(coeff, weight, gap)
    host = api.eval_host(ctx, params, 5, transfer=tables, f_knot0=5e-3, f_knot_step=0.01)
    dev = torch.device("cuda:0")
    ups = torch.empty(n, dtype=torch.float32, device=dev)
    ctx.eval_tf(torch.from_numpy(params).to(dev), 5, torch.from_numpy(tables).to(dev), 4, 5e-3, 0.01, ups)
    torch.cuda.synchronize()
    assert np.array_equal(ups.cpu().numpy(), host["upsilon"])
    with pytest.raises(api.TfsError) as e:
        ctx.eval_tf(params, 5, tables, 4, 5e-3, 0.0, np.empty(n, dtype=np.float32))       # step must be > 0
    assert e.value.code == api.TFS_EINVAL
    with pytest.raises(api.TfsError):
        api.Tfs(w.Nt, w.Nf, w.dt, 4)
    ctx.destroy()
