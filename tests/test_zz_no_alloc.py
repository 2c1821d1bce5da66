"""tfs_topk_static: the top-k entry point for callers that cannot allocate device memory.

Why it exists: tfs_topk (like every other call of the library) lives on a tfs_ctx whose scratch buffers come from
cudaMalloc.  A plug-in running inside a host application that fixed the device-memory budget at start-up, a real-time
loop that cannot take the device-wide synchronisation cudaMalloc/cudaFree imply, or a process whose pool is already
full cannot use that.  tfs_topk_static keeps the select's scratch (radix state + sort keys) in a fixed 514 KiB array
compiled into libtfs.so, takes device pointers only and allocates nothing; the price is the limit
k <= TFS_TOPK_STATIC_MAX_K = 65536 and one shared array per GPU (overlapping calls race).

The file is named test_zz_* so that pytest collects it last: with `pytest -x` a failure here cannot hide another test.
The tests pass alone in a fresh process and after the rest of the suite (they touch no state of other tests: the
static array is used by this entry point only).
"""
import ctypes

import numpy as np
import pytest
import torch

from oracle import tfs_oracle as O


@pytest.fixture(scope="module")
def api():
    from paper_2510_19047_b200 import api as A, build
    build.build()
    return A


def _values(n, seed):
    rng = np.random.default_rng(seed)
    v = rng.chisquare(32, size=n).astype(np.float32)
    v[rng.integers(0, n, size=n // 50)] = v[7]          # ties: equal values must come out in index order
    v[rng.integers(0, n, size=5)] = np.nan               # NaN sorts below everything
    v[rng.integers(0, n, size=5)] = -0.0
    return v


@pytest.mark.gpu
def test_topk_static_matches_tfs_topk_on_two_calls_in_a_row(api):
    """Two calls back to back on one stream, different n and k (the second smaller than the first, so stale keys and a
    stale histogram from call one sit in the shared array when call two starts): both must equal tfs_topk bit for bit
    -- indices exactly, values exactly (top-k is index work; the suite's bar for it is bit-exact) -- and the CPU
    oracle's topk."""
    ctx = api.Tfs(64, 64, 5.0)          # the allocating path, for comparison only
    cases = [(300_001, 10_000, 1), (70_003, 777, 2)]
    ins = [torch.from_numpy(_values(n, seed)).cuda() for n, _, seed in cases]
    outs = []
    for (n, k, _), v in zip(cases, ins):                 # no synchronisation between the two calls
        idx = torch.full((k,), -1, dtype=torch.int64, device="cuda")
        val = torch.full((k,), -1.0, dtype=torch.float32, device="cuda")
        api.topk_static(v, k, idx, val)
        outs.append((idx, val))
    torch.cuda.synchronize()
    for (n, k, _), v, (idx, val) in zip(cases, ins, outs):
        ridx = torch.empty(k, dtype=torch.int64, device="cuda")
        rval = torch.empty(k, dtype=torch.float32, device="cuda")
        ctx.topk(v, k, ridx, rval)
        torch.cuda.synchronize()
        assert torch.equal(idx, ridx), (n, k)
        assert np.array_equal(val.cpu().numpy().view(np.uint32), rval.cpu().numpy().view(np.uint32)), (n, k)
        oi, ov = O.topk(v.cpu().numpy(), k)
        assert np.array_equal(idx.cpu().numpy(), oi), (n, k)
        assert np.array_equal(val.cpu().numpy(), ov.astype(np.float32), equal_nan=True), (n, k)


@pytest.mark.gpu
def test_topk_static_limits_and_small_batches(api):
    """Sizes up to the built-in maximum work (k = 65536 fills the key area exactly); beyond it the call refuses with a
    message that names the limit; host pointers are refused (staging them would need an allocation); a batch small
    enough for the one-launch path (n <= 4096) needs no scratch at all and still agrees."""
    lib = api.load_library()
    ctx = api.Tfs(64, 64, 5.0)
    n, k = 200_000, api.TOPK_STATIC_MAX_K
    v = torch.from_numpy(_values(n, 3)).cuda()
    idx = torch.empty(k, dtype=torch.int64, device="cuda")
    val = torch.empty(k, dtype=torch.float32, device="cuda")
    api.topk_static(v, k, idx, val)
    ridx, rval = torch.empty_like(idx), torch.empty_like(val)
    ctx.topk(v, k, ridx, rval)
    torch.cuda.synchronize()
    assert torch.equal(idx, ridx)
    assert np.array_equal(val.cpu().numpy().view(np.uint32), rval.cpu().numpy().view(np.uint32))

    big = torch.empty(k + 1, dtype=torch.int64, device="cuda")
    bigv = torch.empty(k + 1, dtype=torch.float32, device="cuda")
    with pytest.raises(api.TfsError) as ei:
        api.topk_static(v, k + 1, big, bigv)
    assert ei.value.code == api.TFS_EINVAL and "TFS_TOPK_STATIC_MAX_K" in str(ei.value)

    host = np.zeros(5000, dtype=np.float32)
    hidx, hval = np.zeros(5, dtype=np.int64), np.zeros(5, dtype=np.float32)
    rc = lib.tfs_topk_static(host.ctypes.data, 5000, 5, hidx.ctypes.data, hval.ctypes.data, None)
    assert rc == api.TFS_EINVAL and b"device pointers" in lib.tfs_last_error(None)
    assert lib.tfs_topk_static(None, 10, 1, None, None, None) == api.TFS_EINVAL

    vs = torch.from_numpy(_values(1000, 4)).cuda()
    si = torch.empty(10, dtype=torch.int64, device="cuda")
    sv = torch.empty(10, dtype=torch.float32, device="cuda")
    api.topk_static(vs, 10, si, sv)
    torch.cuda.synchronize()
    oi, ov = O.topk(vs.cpu().numpy(), 10)
    assert np.array_equal(si.cpu().numpy(), oi)
