"""N_seg ladder driver (BASELINE.json configs[4]).

A host loop over the library's calls -- nothing is computed here.  Stage s evaluates its template
set at N_seg = stages[s] (``tfs_eval``), keeps the top ``keep_frac`` (``tfs_topk``) and replaces each
survivor by r x r children on an r-times-denser (Mc, tc) lattice (``tfs_refine``, C19);
the lattice steps shrink by r per stage.  Every array stays on the device between stages.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import torch

from . import api


@dataclass
class Stage:
    N_seg: int
    params: torch.Tensor        # [n][8] float64, device: the templates this stage evaluated
    upsilon: torch.Tensor       # [n] float32, device
    top_idx: torch.Tensor       # [k] int64, device: rows of ``params`` kept, best first
    top_val: torch.Tensor       # [k] float32, device
    d_mc_rel: float             # lattice steps OF THIS STAGE'S templates
    d_tc: float


def run(ctx: api.Tfs, params: torch.Tensor, d_mc_rel: float, d_tc: float, stages=(64, 16, 4, 1),
        keep_frac: float = 0.01, r: int = 4, keep_min: int = 1, stream=None) -> list[Stage]:
    """Run the ladder.  ``params`` [n][8] float64 on the device is the stage-0 bank whose (Mc, tc)
    lattice steps are (Mc*d_mc_rel, d_tc).  Returns one ``Stage`` per entry of ``stages``; the
    last stage's ``top_idx[0]`` row of its ``params`` is the recovered candidate."""
    if not (isinstance(params, torch.Tensor) and params.is_cuda and params.dtype == torch.float64):
        raise TypeError("ladder.run expects a CUDA float64 tensor [n][8]")
    out = []
    cur = params.contiguous()
    for s, N_seg in enumerate(stages):
        n = cur.shape[0]
        ups = torch.empty(n, dtype=torch.float32, device=cur.device)
        ctx.eval(cur, N_seg, ups, stream=stream)
        k = min(n, max(keep_min, int(math.ceil(keep_frac * n))))
        idx = torch.empty(k, dtype=torch.int64, device=cur.device)
        val = torch.empty(k, dtype=torch.float32, device=cur.device)
        ctx.topk(ups, k, idx, val, stream=stream)
        out.append(Stage(N_seg, cur, ups, idx, val, d_mc_rel, d_tc))
        if s + 1 < len(stages):
            nxt = torch.empty((k * r * r, api.PARAM_COLS), dtype=torch.float64, device=cur.device)
            ctx.refine(cur, idx, r, d_mc_rel, d_tc, nxt, stream=stream)
            cur = nxt
            d_mc_rel /= r
            d_tc /= r
    return out
