"""Tile search on the GPU (tfs_tile_lattice, tfs_refine_fin, search.search_tile) against oracle/tfs_search.py
(DESIGN.md section 14).  Lattice positions in M_c are bit-exact; t_c goes through pow on both
sides (a few ulp): 1e-13 relative."""
import numpy as np
import pytest

from oracle import tfs_oracle as O
from oracle import tfs_search as S
from paper_2510_19047_b200 import synth

pytestmark = pytest.mark.gpu

ROW = np.array([0.0, 0.0, 0.7, 0.7, 0.0, 0.5, 0.0, 1.0])


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


def test_tile_lattice_and_refine_fin_match_the_oracle(api):
    import torch
    ctx = api.Tfs(16, 64, 5.0)
    for tile, n_mc, n_fin in (((25.0, 30.0, 8.0e-3, 8.1e-3), 5, 7), ((5.0, 10.0, 2.0e-2, 2.1e-2), 3, 1),
                              ((95.0, 100.0, 1.0e-3, 1.1e-3), 1, 9)):
        ref, d_mc, d_fin = S.tile_lattice(tile[0], tile[1], n_mc, tile[2], tile[3], n_fin, ROW)
        out = np.empty_like(ref)
        ctx.tile_lattice(tile[0], tile[1], n_mc, tile[2], tile[3], n_fin, ROW, out)                 # host output
        assert np.array_equal(out[:, 0], ref[:, 0]) and np.array_equal(out[:, 2:], ref[:, 2:])
        assert np.abs(out[:, 1] / ref[:, 1] - 1).max() < 1e-13
        d_out = torch.empty(ref.shape, dtype=torch.float64, device="cuda")
        ctx.tile_lattice(tile[0], tile[1], n_mc, tile[2], tile[3], n_fin, ROW, d_out)               # device output
        torch.cuda.synchronize()
        assert np.array_equal(d_out.cpu().numpy(), out)
        idx = np.array([len(ref) - 1, 0, len(ref) // 2, 10 ** 6], dtype=np.int64)                  # one out of range
        for r in (1, 3, 4):
            ch_ref = S.refine_fin(ref, idx[:3], r, d_mc, d_fin)
            ch = np.empty((4 * r * r, 8))
            ctx.refine_fin(ref, idx, r, d_mc, d_fin, ch)
            assert np.isnan(ch[3 * r * r:]).all()
            ch = ch[: 3 * r * r]
            assert np.abs(ch[:, 0] - ch_ref[:, 0]).max() <= 1e-14 * 100 and np.array_equal(ch[:, 2:], ch_ref[:, 2:])
            assert np.abs(ch[:, 1] / ch_ref[:, 1] - 1).max() < 1e-12
    with pytest.raises(api.TfsError):
        ctx.tile_lattice(30.0, 25.0, 4, 8e-3, 8.1e-3, 4, ROW, np.empty((16, 8)))
    with pytest.raises(api.TfsError):
        ctx.tile_lattice(25.0, 30.0, 0, 8e-3, 8.1e-3, 4, ROW, np.empty((16, 8)))
    ctx.destroy()


def test_tile_search_recovers_an_injection_like_the_oracle(api):
    """A paper-sized tile (5 Msun x 1e-4 Hz) with one injection in noise: the GPU search and the oracle search
    end on the same candidate (hat-Upsilon_1 within 1e-4, parameters within the final cell), level by level."""
    from paper_2510_19047_b200 import search
    g = O.Grid(48, 256, 40.0)
    rng = np.random.default_rng(21)
    coeff = rng.standard_normal((2, g.Nt, g.Nf, 2)).astype(np.float32)
    Mc, fin = 27.3, 8.037e-3
    inj = ROW.copy(); inj[0] = Mc; inj[1] = float(S.tau_of_f(Mc, fin))
    sig = O.injection(inj, 25.0, None, None, g)
    coeff[..., 0] += sig.real.astype(np.float32)
    coeff[..., 1] += sig.imag.astype(np.float32)
    D = coeff[..., 0].astype(np.float64) + 1j * coeff[..., 1]
    tile = (25.0, 30.0, 8.0e-3, 8.1e-3)
    kw = dict(stages=(4, 1), keep=6, r=3, max_extra=3, tol=1e-3)
    ora = S.search_tile(D, None, None, g, tile, ROW, 6, 12, **kw)
    ctx = api.Tfs(g.Nt, g.Nf, g.dt)
    ctx.upload_data(coeff, None, None)
    gpu = search.search_tile(ctx, tile, ROW, 6, 12, **kw)
    assert len(gpu.levels) == len(ora["levels"])
    for a, b in zip(gpu.levels, ora["levels"]):
        assert a[:2] == b[:2] and abs(a[2] - b[2]) <= 1e-4 * max(b[2], 2.0 * b[0]) and a[3:] == b[3:]
    assert abs(gpu.upsilon - ora["upsilon"]) <= 1e-4 * ora["upsilon"] and gpu.upsilon > 0.85 * 25.0 ** 2
    d_mc_f, d_fin_f = gpu.levels[-1][3], gpu.levels[-1][4]
    assert abs(gpu.params[0] - ora["params"][0]) <= d_mc_f + 1e-12
    assert abs(S.f_of_tau(gpu.params[0], gpu.params[1]) - S.f_of_tau(ora["params"][0], ora["params"][1])) <= d_fin_f + 1e-15
    # a tile 1 mHz (20 bins) away holds no signal: its hat-Upsilon_1 is a noise maximum.  (The neighbour in M_c at the
    # same f_in still sees the source on this 11-day grid: the chirp mass only enters through the slow frequency drift.)
    far = (25.0, 30.0, 9.0e-3, 9.1e-3)
    quiet = search.search_tile(ctx, far, ROW, 6, 12, **kw)
    assert quiet.upsilon < 0.1 * gpu.upsilon
    res = search.search_tiles(ctx, [tile, far], ROW, 6, 12, **kw)
    assert res[0].upsilon == gpu.upsilon and res[1].upsilon == quiet.upsilon           # deterministic
    ctx.destroy()


def test_tile_search_with_a_shared_transfer_table_and_on_a_side_stream(api):
    """search_tile(transfer=...) routes through tfs_eval_tf with one table for the whole tile: a one-knot table holding
    ROW's own (T_A, T_E) must reproduce the plain search (factors applied in fp32 either way); on a 3-channel context it
    is the way to T_T.  With stream= the search runs on that stream (allocations and read-backs ordered with it) and
    returns the same numbers."""
    import torch
    from paper_2510_19047_b200 import search
    g = O.Grid(48, 256, 40.0)
    rng = np.random.default_rng(22)
    coeff = rng.standard_normal((3, g.Nt, g.Nf, 2)).astype(np.float32)
    Mc, fin = 27.3, 8.037e-3
    inj = ROW.copy(); inj[0] = Mc; inj[1] = float(S.tau_of_f(Mc, fin))
    sig = O.injection(inj, 25.0, np.ones((2, g.Nt, g.Nf)), None, g)
    coeff[:2, ..., 0] += sig.real.astype(np.float32)
    coeff[:2, ..., 1] += sig.imag.astype(np.float32)
    tile = (25.0, 30.0, 8.0e-3, 8.1e-3)
    kw = dict(stages=(4, 1), keep=6, r=3, max_extra=2, tol=1e-3)
    ctx = api.Tfs(g.Nt, g.Nf, g.dt)
    ctx.upload_data(np.ascontiguousarray(coeff[:2]), None, None)
    plain = search.search_tile(ctx, tile, ROW, 6, 12, **kw)
    tab2 = np.array([[[ROW[3], ROW[4]]], [[ROW[5], ROW[6]]]], dtype=np.float32)
    with_tab = search.search_tile(ctx, tile, ROW, 6, 12, transfer=(tab2, 0.0, 1.0), **kw)
    assert abs(with_tab.upsilon - plain.upsilon) <= 1e-5 * plain.upsilon and np.array_equal(with_tab.params, plain.params)
    side = torch.cuda.Stream()
    on_side = search.search_tile(ctx, tile, ROW, 6, 12, stream=side.cuda_stream, **kw)
    side.synchronize()
    assert on_side.upsilon == plain.upsilon and np.array_equal(on_side.params, plain.params)
    ctx.destroy()
    # three channels: the plain search is refused until T_T is stated; a table with T_T = 0 equals the 2-channel search
    ctx3 = api.Tfs(g.Nt, g.Nf, g.dt, 3)
    ctx3.upload_data(coeff, None, None)
    with pytest.raises(api.TfsError):
        search.search_tile(ctx3, tile, ROW, 6, 12, **kw)
    tab3 = np.concatenate([tab2, np.zeros((1, 1, 2), dtype=np.float32)])
    three = search.search_tile(ctx3, tile, ROW, 6, 12, transfer=(tab3, 0.0, 1.0), **kw)
    assert abs(three.upsilon - plain.upsilon) <= 1e-5 * plain.upsilon
    tab3[2, 0] = (0.8, 0.1)                                    # noise-only third channel with weight: the statistic moves
    moved = search.search_tile(ctx3, tile, ROW, 6, 12, transfer=(tab3, 0.0, 1.0), **kw)
    assert moved.upsilon != three.upsilon and moved.upsilon > 0.5 * plain.upsilon
    ctx3.destroy()
