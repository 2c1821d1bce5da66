"""CPU fp64 oracle of the search-layer pieces that PAPER.md states without its references
(DESIGN.md section 14).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/`` imports it.  Plain numpy, fp64, no blocking; it
shares no code with the CUDA path and calls ``oracle.tfs_oracle`` for the statistic itself.

What the paper says (P:<line> of PAPER.md):
  P:57   t_0 = 0 at the start of the observation, so the time of coalescence t_c is the remaining lifetime.
  P:269  the search parameters include the chirp mass M_c and f_in = f(t_0), the GW frequency at the start.
  P:275  "we tile the search volume in (M_c, f_in).  Each tile has dimensions of Delta M_c = 5 Msun and
         Delta f_in = 1e-4 (1e-3) Hz for f_in below (above) 1e-2 Hz"; one search per tile.
  P:259  an optimiser identifies "the global maximum of the detection statistic in each parameter tile"
         (a particle swarm whose settings are in refs [30, 59], NOT in the container).
  P:104  "As the search progresses, N_seg is gradually reduced; the final stage, N_seg = 1, is fully coherent".
  P:279  the result of a tile is hat-Upsilon_1 = max over the tile of Upsilon_1.

Readings:
  S1  template model as everywhere else (C5): 0PN, so (M_c, f_in) fixes t_c through the textbook time to
      coalescence  tau(f) = 5 M (8 pi M f)^(-8/3),  M = M_c G Msun / c^3,  t_c = tau(f_in)   (inverse of the track
      f = (tau/5M)^(-3/8)/(8 pi M) of tfs_oracle.track at t = t_0 = 0).
  S2  the optimiser is a deterministic lattice refinement in (M_c, f_in) (the swarm's settings are not available):
      a cell-centred n_mc x n_fin lattice over the tile, then the ladder of BASELINE.json configs[4] (C19) carried
      out in (M_c, f_in): stage s evaluates at N_seg = stages[s], keeps the best ``keep`` rows, and replaces each by
      r x r children on a lattice r times denser per dimension that tiles the parent's cell; the cell shrinks by r
      per stage.
  S3  beyond the fixed ladder: after the last stage the refinement continues at that stage's N_seg around the best
      ``keep`` rows until hat-Upsilon improves by less than ``tol`` (relative) or ``max_extra`` levels were added.
  S4  the other template columns (phase, transfer factors, amplitude) are those of ``row`` for every lattice point
      (the paper also searches sky position, inclination and polarisation through T_alpha; their response functions
      are in ref. [55], not in the container).
"""
from __future__ import annotations

import math

import numpy as np

from oracle import tfs_oracle as O


def tau_of_f(Mc_msun, f):
    """0PN time to coalescence at GW frequency f (S1): tau = 5 M (8 pi M f)^(-8/3)."""
    M = np.asarray(Mc_msun, dtype=np.float64) * O.MTSUN_S
    z = 8.0 * math.pi * M * np.asarray(f, dtype=np.float64)
    return 5.0 * M * z ** (-8.0 / 3.0)


def f_of_tau(Mc_msun, tau):
    """Inverse of tau_of_f: f = (tau / 5M)^(-3/8) / (8 pi M) (the track formula of tfs_oracle.track)."""
    M = np.asarray(Mc_msun, dtype=np.float64) * O.MTSUN_S
    return (np.asarray(tau, dtype=np.float64) / (5.0 * M)) ** (-0.375) / (8.0 * math.pi * M)


def tile_lattice(mc_lo, mc_hi, n_mc: int, fin_lo, fin_hi, n_fin: int, row):
    """Cell-centred lattice over the tile [mc_lo, mc_hi] x [fin_lo, fin_hi] (S2): row i n_fin + j holds
    M_c = mc_lo + (i + 1/2) d_mc, t_c = tau(M_c, fin_lo + (j + 1/2) d_fin), other columns from ``row`` (S4);
    d_mc = (mc_hi - mc_lo)/n_mc, d_fin = (fin_hi - fin_lo)/n_fin.  Returns (params [n_mc n_fin][8], d_mc, d_fin)."""
    row = np.asarray(row, dtype=np.float64)
    d_mc = (np.float64(mc_hi) - np.float64(mc_lo)) / np.float64(n_mc)
    d_fin = (np.float64(fin_hi) - np.float64(fin_lo)) / np.float64(n_fin)
    out = np.empty((n_mc * n_fin, O.PARAM_COLS), dtype=np.float64)
    for i in range(n_mc):
        mc = np.float64(mc_lo) + (np.float64(i) + 0.5) * d_mc
        for j in range(n_fin):
            fin = np.float64(fin_lo) + (np.float64(j) + 0.5) * d_fin
            out[i * n_fin + j] = row
            out[i * n_fin + j, 0] = mc
            out[i * n_fin + j, 1] = tau_of_f(mc, fin)
    return out, float(d_mc), float(d_fin)


def refine_fin(params, idx, r: int, d_mc: float, d_fin: float):
    """r*r children per survivor on a lattice r times denser per dimension that tiles the parent's (M_c, f_in)
    cell of size d_mc x d_fin (S2): o_i = (2i + 1 - r)/(2r); child (a, b) of parent j at row j r^2 + a r + b:
    M_c' = M_c + o_a d_mc,  f_in' = f_in + o_b d_fin with f_in = f_of_tau(M_c, t_c),  t_c' = tau(M_c', f_in')."""
    params = np.asarray(params, dtype=np.float64)
    out = np.empty((len(idx) * r * r, O.PARAM_COLS), dtype=np.float64)
    row = 0
    for j in idx:
        p = params[int(j)]
        fin = f_of_tau(p[0], p[1])
        for a in range(r):
            oa = np.float64(2 * a + 1 - r) / np.float64(2 * r)
            for b in range(r):
                ob = np.float64(2 * b + 1 - r) / np.float64(2 * r)
                mc = p[0] + oa * d_mc
                out[row] = p
                out[row, 0] = mc
                out[row, 1] = tau_of_f(mc, fin + ob * d_fin)
                row += 1
    return out


def search_tile(D, W, gap_mask, grid: O.Grid, tile, row, n_mc: int, n_fin: int, stages=(16, 4, 1), keep: int = 8,
                r: int = 4, max_extra: int = 3, tol: float = 1e-3, opts: O.Opts = O.Opts()):
    """Search one tile (mc_lo, mc_hi, fin_lo, fin_hi) (S2, S3).  Returns dict(upsilon = hat-Upsilon at the last
    N_seg, params = its row, levels = [(N_seg, n_evaluated, best Upsilon, d_mc, d_fin)])."""
    cur, d_mc, d_fin = tile_lattice(tile[0], tile[1], n_mc, tile[2], tile[3], n_fin, row)
    levels = []
    best_u, best_p = -1.0, None
    n_levels = len(stages) + max_extra
    for lev in range(n_levels):
        N_seg = stages[min(lev, len(stages) - 1)]
        ups = O.evaluate(cur, D, W, gap_mask, grid, N_seg, opts)["upsilon"]
        idx, val = O.topk(ups, min(len(cur), keep))
        levels.append((N_seg, len(cur), float(val[0]), d_mc, d_fin))
        if lev >= len(stages) - 1:                       # levels at the final N_seg: track hat-Upsilon (S3)
            gain = float(val[0]) > best_u * (1.0 + tol)
            if float(val[0]) > best_u:
                best_u, best_p = float(val[0]), cur[int(idx[0])].copy()
            if lev > len(stages) - 1 and not gain:
                break
        if lev + 1 < n_levels:
            cur = refine_fin(cur, idx, r, d_mc, d_fin)
            d_mc /= r
            d_fin /= r
    return dict(upsilon=best_u, params=best_p, levels=levels)
