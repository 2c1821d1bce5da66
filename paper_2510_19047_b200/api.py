"""Thin Python binding of libtfs (include/tfs.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used here only to own
device memory and to name the current stream.  There is no fallback: if ``libtfs.so`` is
missing or no CUDA device is present these calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("TFS_LIB_PATH") or os.path.join(_HERE, "libtfs.so")   # override: A/B-testing builds

TFS_OK, TFS_EINVAL, TFS_ESTATE, TFS_ENOMEM, TFS_ECUDA = 0, -1, -2, -3, -4
PARAM_COLS = 8


class tfs_opts(C.Structure):
    _fields_ = [("half_width", C.c_int), ("adaptive_width", C.c_int), ("c_max", C.c_double),
                ("f_lo", C.c_double), ("f_hi", C.c_double), ("fresnel_mode", C.c_int),
                ("weight_mode", C.c_int), ("basis", C.c_int), ("wdm_half_width", C.c_int),
                ("wdm_kappa_max", C.c_double), ("tukey_alpha", C.c_double)]


class TfsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libtfs error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libtfs.so (built in-tree by ``python -m paper_2510_19047_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2510_19047_b200.build` "
                           "(libtfs has no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, ip, dp, ll = C.c_void_p, C.c_int, C.c_double, C.c_longlong
    lib.tfs_default_opts.argtypes = [C.POINTER(tfs_opts)]
    lib.tfs_default_opts.restype = None
    lib.tfs_create.argtypes = [C.POINTER(vp), ip, ip, dp, ip, C.POINTER(tfs_opts)]
    lib.tfs_create.restype = ip
    lib.tfs_upload_data.argtypes = [vp, vp, vp, vp, vp]
    lib.tfs_upload_data.restype = ip
    lib.tfs_upload_timeseries.argtypes = [vp, vp, vp, vp, dp, vp, vp, vp, vp]
    lib.tfs_upload_timeseries.restype = ip
    lib.tfs_eval.argtypes = [vp, vp, ll, ip, vp, vp, vp, vp, vp]
    lib.tfs_eval.restype = ip
    lib.tfs_eval_tf.argtypes = [vp, vp, ll, ip, vp, ip, dp, dp, vp, vp, vp, vp, vp]
    lib.tfs_eval_tf.restype = ip
    lib.tfs_eval_tseg.argtypes = [vp, vp, ll, ip, vp, vp, vp, vp, vp, vp]
    lib.tfs_eval_tseg.restype = ip
    lib.tfs_topk.argtypes = [vp, vp, ll, ip, vp, vp, vp]
    lib.tfs_topk.restype = ip
    lib.tfs_set_third_channel_factor.argtypes = [vp, dp, dp]
    lib.tfs_set_third_channel_factor.restype = ip
    lib.tfs_topk_static.argtypes = [vp, ll, ip, vp, vp, vp]
    lib.tfs_topk_static.restype = ip
    lib.tfs_refine.argtypes = [vp, vp, ll, vp, ll, ip, dp, dp, vp, vp]
    lib.tfs_refine.restype = ip
    lib.tfs_refine_fin.argtypes = [vp, vp, ll, vp, ll, ip, dp, dp, vp, vp]
    lib.tfs_refine_fin.restype = ip
    lib.tfs_tile_lattice.argtypes = [vp, dp, dp, ip, dp, dp, ip, vp, vp, vp]
    lib.tfs_tile_lattice.restype = ip
    lib.tfs_count_pixels.argtypes = [vp, vp, ll, vp, vp]
    lib.tfs_count_pixels.restype = ip
    lib.tfs_bad_param_count.argtypes = [vp]
    lib.tfs_bad_param_count.restype = ll
    lib.tfs_weight_structure.argtypes = [vp]
    lib.tfs_weight_structure.restype = ip
    lib.tfs_set_profiling.argtypes = [vp, ip]
    lib.tfs_set_profiling.restype = ip
    lib.tfs_get_profile.argtypes = [vp, C.POINTER(dp), C.POINTER(ll), C.POINTER(ll)]
    lib.tfs_get_profile.restype = ip
    lib.tfs_get_profile_kernels.argtypes = [vp, C.POINTER(dp), C.POINTER(dp), C.POINTER(ll), C.POINTER(ll)]
    lib.tfs_get_profile_kernels.restype = ip
    lib.tfs_probe_fp32_issue.argtypes = [vp, ip, C.POINTER(dp), C.POINTER(dp), vp]
    lib.tfs_probe_fp32_issue.restype = ip
    lib.tfs_tier_census.argtypes = [vp, ip, C.POINTER(ll)]
    lib.tfs_tier_census.restype = ip
    lib.tfs_probe_l2_bandwidth.argtypes = [vp, ll, ip, C.POINTER(dp), vp]
    lib.tfs_probe_l2_bandwidth.restype = ip
    lib.tfs_destroy.argtypes = [vp]
    lib.tfs_destroy.restype = None
    lib.tfs_last_error.argtypes = [vp]
    lib.tfs_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _ptr(x, dtype, nelem=None):
    """Raw address of a contiguous numpy array or torch tensor of the given dtype (or None)."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if x.dtype != np.dtype(dtype) or not x.flags["C_CONTIGUOUS"]:
            raise TypeError(f"expected C-contiguous {np.dtype(dtype)} array, got {x.dtype}")
        if nelem is not None and x.size < nelem:
            raise ValueError(f"array too small: {x.size} < {nelem}")
        return x.ctypes.data
    import torch
    if isinstance(x, torch.Tensor):
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int64: torch.int64,
                np.int32: torch.int32, np.uint8: torch.uint8}[dtype]
        if x.dtype != want or not x.is_contiguous():
            raise TypeError(f"expected contiguous {want} tensor, got {x.dtype}")
        if nelem is not None and x.numel() < nelem:
            raise ValueError(f"tensor too small: {x.numel()} < {nelem}")
        return x.data_ptr()
    raise TypeError(f"unsupported buffer type {type(x)}")


def _stream(stream):
    if stream is not None:
        return int(stream)
    import torch
    return torch.cuda.current_stream().cuda_stream


class Tfs:
    """One libtfs context (``tfs_ctx``).  Methods carry the C names without the prefix."""

    def __init__(self, Nt, Nf, dt, n_channels=2, **opts):
        self._lib = load_library()
        o = tfs_opts()
        self._lib.tfs_default_opts(C.byref(o))
        for k, v in opts.items():
            if not hasattr(o, k):
                raise TypeError(f"unknown option {k}")
            setattr(o, k, v)
        h = C.c_void_p()
        rc = self._lib.tfs_create(C.byref(h), Nt, Nf, dt, n_channels, C.byref(o))
        if rc != TFS_OK:
            raise TfsError(rc, self._lib.tfs_last_error(None).decode())
        self._h = h
        self.Nt, self.Nf, self.dt, self.C = Nt, Nf, dt, n_channels
        self.basis = int(o.basis)

    def _check(self, rc):
        if rc != TFS_OK:
            raise TfsError(rc, self._lib.tfs_last_error(self._h).decode())

    def upload_data(self, coeff, weight=None, gap_mask=None, stream=None):
        npix = self.C * self.Nt * self.Nf
        self._check(self._lib.tfs_upload_data(self._h, _ptr(coeff, np.float32, (1 if self.basis == 1 else 2) * npix),
                                              _ptr(weight, np.float32, npix),
                                              _ptr(gap_mask, np.uint8, self.Nt), _stream(stream)))

    def upload_timeseries(self, x, sample_mask=None, psd=None, tukey_alpha=0.1, coeff_out=None, weight_out=None,
                          gap_out=None, stream=None):
        nsamp = self.Nt * 2 * self.Nf
        npix = self.C * self.Nt * self.Nf
        self._check(self._lib.tfs_upload_timeseries(
            self._h, _ptr(x, np.float32, self.C * nsamp), _ptr(sample_mask, np.uint8, nsamp),
            _ptr(psd, np.float32, self.C * self.Nf), float(tukey_alpha), _ptr(coeff_out, np.float32, 2 * npix),
            _ptr(weight_out, np.float32, npix), _ptr(gap_out, np.uint8, self.Nt), _stream(stream)))

    def eval(self, params, N_seg, upsilon, seg_power=None, seg_dh=None, seg_hh=None, n=None, stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        self._check(self._lib.tfs_eval(self._h, _ptr(params, np.float64, n * PARAM_COLS), n, N_seg,
                                       _ptr(upsilon, np.float32, n), _ptr(seg_power, np.float32, n * N_seg),
                                       _ptr(seg_dh, np.float32, 2 * n * N_seg),
                                       _ptr(seg_hh, np.float32, n * N_seg), _stream(stream)))

    def eval_tseg(self, params, seg_tranches, upsilon, n_seg_eff=None, seg_power=None, seg_dh=None, seg_hh=None, n=None,
                  stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        N_seg = -(-self.Nt // max(int(seg_tranches), 1))
        self._check(self._lib.tfs_eval_tseg(self._h, _ptr(params, np.float64, n * PARAM_COLS), n, seg_tranches,
                                            _ptr(upsilon, np.float32, n), _ptr(n_seg_eff, np.int32, n),
                                            _ptr(seg_power, np.float32, n * N_seg), _ptr(seg_dh, np.float32, 2 * n * N_seg),
                                            _ptr(seg_hh, np.float32, n * N_seg), _stream(stream)))

    def eval_tf(self, params, N_seg, transfer, n_knots, f_knot0, f_knot_step, upsilon, seg_power=None, seg_dh=None,
                seg_hh=None, n=None, stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        self._check(self._lib.tfs_eval_tf(self._h, _ptr(params, np.float64, n * PARAM_COLS), n, N_seg,
                                          _ptr(transfer, np.float32, 2 * n * self.C * n_knots), n_knots,
                                          float(f_knot0), float(f_knot_step),
                                          _ptr(upsilon, np.float32, n), _ptr(seg_power, np.float32, n * N_seg),
                                          _ptr(seg_dh, np.float32, 2 * n * N_seg),
                                          _ptr(seg_hh, np.float32, n * N_seg), _stream(stream)))

    def probe_fp32_issue(self, iters=1 << 16, stream=None):
        """tfs_probe_fp32_issue: (scalar FFMA, packed FFMA2) warp instructions per clock per SM."""
        a, b = C.c_double(), C.c_double()
        self._check(self._lib.tfs_probe_fp32_issue(self._h, int(iters), C.byref(a), C.byref(b), _stream(stream)))
        return a.value, b.value

    def tier_census(self, on):
        """tfs_tier_census: returns the five tier counters accumulated since the previous call, then switches the census on/off."""
        out = (C.c_longlong * 5)()
        self._check(self._lib.tfs_tier_census(self._h, int(bool(on)), out))
        return [int(v) for v in out]

    def set_third_channel_factor(self, re, im=0.0):
        self._check(self._lib.tfs_set_third_channel_factor(self._h, float(re), float(im)))

    def topk(self, upsilon, k, idx, val, n=None, stream=None):
        if n is None:
            n = upsilon.size if isinstance(upsilon, np.ndarray) else upsilon.numel()
        self._check(self._lib.tfs_topk(self._h, _ptr(upsilon, np.float32, n), n, k,
                                       _ptr(idx, np.int64, k), _ptr(val, np.float32, k), _stream(stream)))

    def refine(self, params, idx, r, d_mc_rel, d_tc, children, n=None, k=None, stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        if k is None:
            k = idx.size if isinstance(idx, np.ndarray) else idx.numel()
        self._check(self._lib.tfs_refine(self._h, _ptr(params, np.float64, n * PARAM_COLS), n,
                                         _ptr(idx, np.int64, k), k, r, d_mc_rel, d_tc,
                                         _ptr(children, np.float64, k * r * r * PARAM_COLS), _stream(stream)))

    def refine_fin(self, params, idx, r, d_mc, d_fin, children, n=None, k=None, stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        if k is None:
            k = idx.size if isinstance(idx, np.ndarray) else idx.numel()
        self._check(self._lib.tfs_refine_fin(self._h, _ptr(params, np.float64, n * PARAM_COLS), n,
                                             _ptr(idx, np.int64, k), k, r, d_mc, d_fin,
                                             _ptr(children, np.float64, k * r * r * PARAM_COLS), _stream(stream)))

    def tile_lattice(self, mc_lo, mc_hi, n_mc, fin_lo, fin_hi, n_fin, row, params, stream=None):
        row = np.ascontiguousarray(row, dtype=np.float64)
        if row.size != PARAM_COLS:
            raise ValueError("row must hold 8 doubles")
        self._check(self._lib.tfs_tile_lattice(self._h, mc_lo, mc_hi, n_mc, fin_lo, fin_hi, n_fin, row.ctypes.data,
                                               _ptr(params, np.float64, n_mc * n_fin * PARAM_COLS), _stream(stream)))

    def count_pixels(self, params, counts, n=None, stream=None):
        if n is None:
            n = (params.size if isinstance(params, np.ndarray) else params.numel()) // PARAM_COLS
        self._check(self._lib.tfs_count_pixels(self._h, _ptr(params, np.float64, n * PARAM_COLS), n,
                                               _ptr(counts, np.int64, n), _stream(stream)))

    def bad_param_count(self):
        return int(self._lib.tfs_bad_param_count(self._h))

    def weight_structure(self):
        return int(self._lib.tfs_weight_structure(self._h))

    def set_profiling(self, on=True):
        self._check(self._lib.tfs_set_profiling(self._h, int(bool(on))))

    def get_profile(self):
        ms, nk, nl = C.c_double(), C.c_longlong(), C.c_longlong()
        self._check(self._lib.tfs_get_profile(self._h, C.byref(ms), C.byref(nk), C.byref(nl)))
        return dict(main_kernel_ms=ms.value, main_kernel_launches=nk.value, kernel_launches=nl.value)

    def get_profile_kernels(self):
        a, b, nk, nl = C.c_double(), C.c_double(), C.c_longlong(), C.c_longlong()
        self._check(self._lib.tfs_get_profile_kernels(self._h, C.byref(a), C.byref(b), C.byref(nk), C.byref(nl)))
        return dict(slab_kernel_ms=a.value, list_kernel_ms=b.value, eval_launches=nk.value, kernel_launches=nl.value)

    def probe_l2_bandwidth(self, nbytes=32 << 20, iters=200, stream=None):
        g = C.c_double()
        self._check(self._lib.tfs_probe_l2_bandwidth(self._h, nbytes, iters, C.byref(g), _stream(stream)))
        return g.value

    def last_error(self):
        return self._lib.tfs_last_error(self._h).decode()

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.tfs_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ---- convenience wrappers on host numpy buffers (used by tests, smoke and the e2e bench leg) ----
def eval_host(ctx: Tfs, params: np.ndarray, N_seg: int, segments: bool = True, transfer=None, f_knot0=0.0,
              f_knot_step=1.0):
    """tfs_eval (or tfs_eval_tf when a transfer table [n][C][K][2] is given) with HOST buffers in and out
    (the library does the copies)."""
    params = np.ascontiguousarray(params, dtype=np.float64)
    n = params.shape[0]
    ups = np.empty(n, dtype=np.float32)
    if transfer is not None:
        transfer = np.ascontiguousarray(transfer, dtype=np.float32)
        K = transfer.shape[2]

        def run(*out):
            ctx.eval_tf(params, N_seg, transfer, K, f_knot0, f_knot_step, *out)
    else:
        def run(*out):
            ctx.eval(params, N_seg, *out)
    if not segments:
        run(ups)
        return dict(upsilon=ups)
    P = np.empty((n, N_seg), dtype=np.float32)
    z = np.empty((n, N_seg, 2), dtype=np.float32)
    hh = np.empty((n, N_seg), dtype=np.float32)
    run(ups, P, z, hh)
    return dict(upsilon=ups, seg_power=P, seg_dh=z[..., 0] + 1j * z[..., 1], seg_hh=hh)


def topk_host(ctx: Tfs, upsilon: np.ndarray, k: int):
    upsilon = np.ascontiguousarray(upsilon, dtype=np.float32)
    idx = np.empty(k, dtype=np.int64)
    val = np.empty(k, dtype=np.float32)
    ctx.topk(upsilon, k, idx, val)
    return idx, val


TOPK_STATIC_MAX_K = 65536       # TFS_TOPK_STATIC_MAX_K of include/tfs.h


def topk_static(upsilon, k, idx, val, n=None, stream=None):
    """``tfs_topk_static``: the top-k of ``tfs_topk`` for callers that are not allowed to allocate device memory
    (a plug-in living inside someone else's fixed memory budget, a latency-critical loop that cannot take the
    device-wide stall of ``cudaMalloc``/``cudaFree``, a process whose pool is full).  No context is needed; the
    select's scratch is a 514 KiB array built into ``libtfs.so``.  ``upsilon``, ``idx`` (int64) and ``val`` (float32)
    must be CUDA tensors on the current device and ``k <= TOPK_STATIC_MAX_K``; anything else raises ``TfsError``
    (``TFS_EINVAL``).  Only enqueues on ``stream``.  All calls on one GPU share that one array: issue them in order
    on one stream (or order them with events) -- overlapping calls corrupt each other's result.  The first call
    on a device also looks up the array's address; do it before starting any stream capture."""
    lib = load_library()
    if n is None:
        n = upsilon.numel()
    rc = lib.tfs_topk_static(_ptr(upsilon, np.float32, n), n, k, _ptr(idx, np.int64, min(k, max(n, 0))),
                             _ptr(val, np.float32, min(k, max(n, 0))), _stream(stream))
    if rc != TFS_OK:
        raise TfsError(rc, lib.tfs_last_error(None).decode())


def eval_tseg_host(ctx: Tfs, params: np.ndarray, seg_tranches: int):
    """tfs_eval_tseg with HOST buffers in and out."""
    params = np.ascontiguousarray(params, dtype=np.float64)
    n = params.shape[0]
    N_seg = -(-ctx.Nt // max(int(seg_tranches), 1))
    ups = np.empty(n, dtype=np.float32)
    neff = np.empty(n, dtype=np.int32)
    P = np.empty((n, N_seg), dtype=np.float32)
    z = np.empty((n, N_seg, 2), dtype=np.float32)
    hh = np.empty((n, N_seg), dtype=np.float32)
    ctx.eval_tseg(params, seg_tranches, ups, neff, P, z, hh)
    return dict(upsilon=ups, n_seg_eff=neff, seg_power=P, seg_dh=z[..., 0] + 1j * z[..., 1], seg_hh=hh)
