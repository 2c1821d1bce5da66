"""Per-tile search driver (P:275 tiles in (Mc, f_in), P:259 one
maximisation per tile, P:104 N_seg reduced stage by stage, P:279 hat-Upsilon_1 per tile).

A host loop over the library's calls -- nothing is computed here.  Level 0 evaluates the tile's cell-centred
(Mc, f_in) lattice (``tfs_tile_lattice``) at N_seg = stages[0]; every level keeps the best ``keep`` rows
(``tfs_topk``) and replaces each by r x r children that tile its cell (``tfs_refine_fin``); after the last stage
the refinement continues at that N_seg until hat-Upsilon gains less than ``tol`` (relative) or ``max_extra`` extra
levels were added (readings S2, S3).  Every array stays on the device; one float and one row are read back per level.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

from . import api


@dataclass
class TileResult:
    upsilon: float                       # hat-Upsilon at the final N_seg
    params: np.ndarray                   # [8] the row that reached it
    levels: list = field(default_factory=list)   # (N_seg, n_evaluated, best Upsilon, d_mc, d_fin) per level


def search_tile(ctx: api.Tfs, tile, row, n_mc: int, n_fin: int, stages=(16, 4, 1), keep: int = 8, r: int = 4,
                max_extra: int = 3, tol: float = 1e-3, stream=None, transfer=None) -> TileResult:
    """tile = (mc_lo, mc_hi, fin_lo, fin_hi) in Msun and Hz; ``row`` [8] gives the columns the lattice does not span.

    ``transfer`` = (table [C][K][2] float32, f_knot0, f_knot_step): one transfer table shared by every template of the
    tile (sky position and polarisation are fixed by ``row``), evaluated with ``tfs_eval_tf`` -- the way a 3-channel
    context gets its T_T(f); without it the search calls ``tfs_eval`` (on a 3-channel context that needs
    ``set_third_channel_factor`` first).

    ``stream``: a raw CUDA stream handle.  The whole search -- library calls, the tensors allocated here and the two
    scalars read back per level -- then runs with that stream as torch's current stream, so the caching allocator and
    the ``.item()`` reads are ordered with the library's kernels."""
    if stream is not None:
        with torch.cuda.stream(torch.cuda.ExternalStream(int(stream))):
            return search_tile(ctx, tile, row, n_mc, n_fin, stages, keep, r, max_extra, tol, None, transfer)
    dev = torch.device("cuda", torch.cuda.current_device())
    tab = None
    if transfer is not None:
        tab, f_knot0, f_knot_step = transfer
        tab = torch.as_tensor(np.ascontiguousarray(tab, dtype=np.float32) if isinstance(tab, np.ndarray) else tab,
                              device=dev).to(torch.float32)
        n_knots = int(tab.shape[1])
    mc_lo, mc_hi, fin_lo, fin_hi = (float(v) for v in tile)
    d_mc, d_fin = (mc_hi - mc_lo) / n_mc, (fin_hi - fin_lo) / n_fin
    cur = torch.empty((n_mc * n_fin, api.PARAM_COLS), dtype=torch.float64, device=dev)
    ctx.tile_lattice(mc_lo, mc_hi, n_mc, fin_lo, fin_hi, n_fin, row, cur, stream=stream)
    res = TileResult(-1.0, np.zeros(api.PARAM_COLS))
    n_levels = len(stages) + max_extra
    for lev in range(n_levels):
        N_seg = stages[min(lev, len(stages) - 1)]
        n = cur.shape[0]
        ups = torch.empty(n, dtype=torch.float32, device=dev)
        if tab is None:
            ctx.eval(cur, N_seg, ups, stream=stream)
        else:
            ctx.eval_tf(cur, N_seg, tab.unsqueeze(0).expand(n, *tab.shape).contiguous(), n_knots, float(f_knot0),
                        float(f_knot_step), ups, stream=stream)
        k = min(n, keep)
        idx = torch.empty(k, dtype=torch.int64, device=dev)
        val = torch.empty(k, dtype=torch.float32, device=dev)
        ctx.topk(ups, k, idx, val, stream=stream)
        top = float(val[0].item())
        res.levels.append((N_seg, n, top, d_mc, d_fin))
        if lev >= len(stages) - 1:
            gain = top > res.upsilon * (1.0 + tol)
            if top > res.upsilon:
                res.upsilon = top
                res.params = cur[int(idx[0].item())].cpu().numpy()
            if lev > len(stages) - 1 and not gain:
                break
        if lev + 1 < n_levels:
            nxt = torch.empty((k * r * r, api.PARAM_COLS), dtype=torch.float64, device=dev)
            ctx.refine_fin(cur, idx, r, d_mc, d_fin, nxt, stream=stream)
            cur = nxt
            d_mc /= r
            d_fin /= r
    return res


def search_tiles(ctx: api.Tfs, tiles, row, n_mc: int, n_fin: int, **kw):
    """hat-Upsilon per tile (the map of Fig. 4, top left): a list of TileResult, one per (mc_lo, mc_hi, fin_lo, fin_hi)."""
    return [search_tile(ctx, t, row, n_mc, n_fin, **kw) for t in tiles]
