"""Pins of the search-layer oracle (oracle/tfs_search.py).  CPU only."""
import math

import numpy as np

from oracle import tfs_oracle as O
from oracle import tfs_search as S


# S-1  t_c = tau(M_c, f_in) is the inverse of the track: a template built from (M_c, f_in) starts at f_in
#      (P:57 t_0 = 0 so that t_c is the remaining lifetime; P:269 f_in = f(t_0)); textbook numbers
def test_s1_tau_is_the_inverse_of_the_track():
    g = O.Grid(8, 64, 5.0)
    for Mc in (5.0, 30.0, 100.0):
        for fin in (1e-3, 8e-3, 3e-2, 0.1):
            tc = float(S.tau_of_f(Mc, fin))
            tr = O.track(Mc, tc, 0.0, 1.0, g, O.Opts(f_lo=0.0, f_hi=1e9, c_max=1e300))
            assert abs(tr["f"][0] / fin - 1.0) < 1e-13                     # tranche 0 starts at t_0 = 0
            assert abs(float(S.f_of_tau(Mc, tc)) / fin - 1.0) < 1e-13
    # tau ~ f^(-8/3) M_c^(-5/3): scaling, and the survey's appendix value (M_c = 30, t_c = 1 yr starts at 27.8 mHz)
    assert abs(float(S.tau_of_f(30.0, 2e-2) / S.tau_of_f(30.0, 1e-2)) - 2.0 ** (-8.0 / 3.0)) < 1e-14
    assert abs(float(S.tau_of_f(60.0, 1e-2) / S.tau_of_f(30.0, 1e-2)) - 2.0 ** (-5.0 / 3.0)) < 1e-14
    assert abs(float(S.f_of_tau(30.0, O.YEAR_S)) - 27.8e-3) < 0.05e-3


# S-2  the lattice is cell-centred and covers the tile evenly; the paper's tile sizes
def test_s2_tile_lattice():
    row = np.array([0.0, 0.0, 0.4, 0.7, 0.1, 0.5, -0.2, 1.5])
    p, d_mc, d_fin = S.tile_lattice(25.0, 30.0, 5, 8.0e-3, 8.1e-3, 4, row)
    assert p.shape == (20, 8) and d_mc == 1.0 and abs(d_fin - 2.5e-5) < 1e-18
    assert np.array_equal(p[:, 2:], np.broadcast_to(row[2:], (20, 6)))
    mc = p[:, 0].reshape(5, 4)
    assert np.array_equal(mc[:, 0], [25.5, 26.5, 27.5, 28.5, 29.5]) and (mc == mc[:, :1]).all()
    fin = S.f_of_tau(p[:, 0], p[:, 1]).reshape(5, 4)
    assert np.allclose(fin, 8.0e-3 + (np.arange(4) + 0.5) * 2.5e-5, rtol=1e-13, atol=0)
    assert (np.diff(p[:, 1].reshape(5, 4), axis=1) < 0).all()             # higher f_in merges sooner


# S-3  children tile the parent's cell: refining every point of a regular lattice gives one regular lattice of step d/r
def test_s3_children_tile_the_parent_cell():
    row = np.array([0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0])
    for r in (1, 2, 3, 4):
        p, d_mc, d_fin = S.tile_lattice(20.0, 24.0, 4, 5e-3, 6e-3, 5, row)
        ch = S.refine_fin(p, np.arange(len(p)), r, d_mc, d_fin)
        assert ch.shape == (len(p) * r * r, 8)
        mcs = np.unique(np.round(ch[:, 0], 9))
        fins = np.unique(np.round(S.f_of_tau(ch[:, 0], ch[:, 1]), 12))
        assert len(mcs) == 4 * r and np.allclose(np.diff(mcs), d_mc / r, rtol=1e-9)
        assert len(fins) == 5 * r and np.allclose(np.diff(fins), d_fin / r, rtol=1e-6)
        assert abs(mcs[0] - (20.0 + d_mc / (2 * r))) < 1e-9 and abs(fins[0] - (5e-3 + d_fin / (2 * r))) < 1e-12
    # r = 1 returns the parents (up to the round trip t_c -> f_in -> t_c)
    ch = S.refine_fin(p, [3, 0], 1, d_mc, d_fin)
    assert np.allclose(ch, p[[3, 0]], rtol=1e-13, atol=0)


# S-4  a noiseless injection inside a tile is found: hat-Upsilon_1 > 0.9 rho^2, parameters within two final cells,
#      while the coarse lattice alone scores far below; the extra levels (S3) stop on their own
def test_s4_tile_search_recovers_an_injection():
    g = O.Grid(48, 256, 40.0)                       # DT = 20480 s, T_obs = 11.4 d, df = 48.8 uHz
    Mc, fin = 27.3, 8.037e-3
    tc = float(S.tau_of_f(Mc, fin))
    inj = np.array([Mc, tc, 0.7, 0.7, 0.0, 0.5, 0.0, 1.0])
    rho = 30.0
    D = O.injection(inj, rho, None, None, g)
    row = inj.copy(); row[0] = 0.0; row[1] = 0.0
    tile = (25.0, 30.0, 8.0e-3, 8.1e-3)             # the paper's tile: 5 Msun x 1e-4 Hz below 10 mHz
    res = S.search_tile(D, None, None, g, tile, row, 6, 12, stages=(4, 1), keep=6, r=3, max_extra=4, tol=1e-3)
    lv = res["levels"]
    assert [l[0] for l in lv[:2]] == [4, 1] and all(l[0] == 1 for l in lv[2:]) and 3 <= len(lv) <= 6
    assert res["upsilon"] > 0.9 * rho ** 2, res["upsilon"] / rho ** 2
    d_mc_f, d_fin_f = lv[-1][3], lv[-1][4]
    fin_rec = float(S.f_of_tau(res["params"][0], res["params"][1]))
    assert abs(fin_rec - fin) < 2 * max(d_fin_f, 1e-9)
    # the coarse lattice alone is far from the peak at N_seg = 1
    coarse, _, _ = S.tile_lattice(*tile[:2], 6, *tile[2:], 12, row)
    u0 = O.evaluate(coarse, D, None, None, g, 1)["upsilon"].max()
    assert u0 < 0.75 * res["upsilon"]
    # hat-Upsilon never decreases along the levels at N_seg = 1
    best = np.maximum.accumulate([l[2] for l in lv[1:]])
    assert res["upsilon"] == best[-1]


# S-5  an empty tile (noise only): the search returns the largest noise fluctuation, a finite number well below an
#      injection's, and respects max_extra
def test_s5_noise_only_tile():
    rng = np.random.default_rng(5)
    g = O.Grid(32, 128, 40.0)
    D = rng.standard_normal((2, g.Nt, g.Nf)) + 1j * rng.standard_normal((2, g.Nt, g.Nf))
    row = np.array([0.0, 0.0, 0.0, 0.7, 0.0, 0.5, 0.0, 1.0])
    res = S.search_tile(D, None, None, g, (25.0, 30.0, 8.0e-3, 8.1e-3), row, 3, 4, stages=(2, 1), keep=3, r=2,
                        max_extra=2, tol=1e-2)
    assert len(res["levels"]) <= 4 and 0.0 < res["upsilon"] < 40.0 and np.isfinite(res["params"]).all()
    assert math.isclose(res["levels"][0][3], 5.0 / 3) and res["levels"][1][1] == 3 * 4
