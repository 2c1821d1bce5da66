"""The measurement hooks bench.py's roofline uses: tfs_tier_census (pixel slots evaluated per tier) and
tfs_probe_fp32_issue (FP32 issue rate of one SM).  They must not change any result."""
import numpy as np
import pytest

from paper_2510_19047_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as _api, build
    build.build()
    return _api


def test_tier_census_counts_every_window_pixel_and_changes_nothing(api):
    import torch
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=700, Nf=1024, n_templates=3000)
    coeff, weight, gap = synth.make_data(w)
    params = synth.make_templates(w)
    ctx = api.Tfs(w.Nt, w.Nf, w.dt)
    ctx.upload_data(coeff, weight, gap)
    d = torch.from_numpy(params).cuda()
    n = len(params)
    counts = torch.empty(n, dtype=torch.int64, device="cuda")
    ctx.count_pixels(d, counts)
    pixels = int(counts.sum().item())
    ups0 = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.eval(d, 7, ups0)
    assert ctx.tier_census(True) == [0, 0, 0, 0, 0]              # nothing is counted while the census is off
    ups1 = torch.empty_like(ups0)
    ctx.eval(d, 7, ups1)
    c = ctx.tier_census(True)
    ctx.eval(d, 7, ups1)
    c2 = ctx.tier_census(False)
    assert c == c2 and all(v >= 0 for v in c)                     # deterministic, and zeroed by every read
    assert torch.equal(ups0, ups1)                                # counting changes no result
    total = sum(c)
    # every window pixel is evaluated in exactly one tier; the rest of the slots are padding (inactive lanes,
    # windows shorter than the warp's longest), bounded by the tile geometry
    assert pixels <= total <= 4 * pixels, (pixels, c)
    assert c[0] + c[1] + c[3] > 0 and c[2] + c[4] > 0            # far and near tiers both occur on this bank
    assert c[0] % 64 == 0 and c[1] % 64 == 0 and c[2] % 64 == 0 and c[3] % 32 == 0 and c[4] % 32 == 0
    ctx.eval(d, 7, ups1)
    assert ctx.tier_census(False) == [0, 0, 0, 0, 0]
    ctx.destroy()


def test_fp32_issue_probe_is_within_the_hardware_limits(api):
    ctx = api.Tfs(16, 64, 5.0)
    scalar, packed = ctx.probe_fp32_issue(1 << 14)
    # four schedulers issue at most one warp instruction per clock each; a packed FFMA2 occupies the pipe for two
    assert 2.0 < scalar <= 4.05 and 1.0 < packed <= 2.05, (scalar, packed)
    with pytest.raises(api.TfsError):
        ctx.probe_fp32_issue(0)
    ctx.destroy()
