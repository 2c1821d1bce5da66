"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/tfs.h declares.
No compute calls: runs without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2510_19047_b200 import build
    return build.build()


def declared_symbols():
    h = open(os.path.join(ROOT, "include", "tfs.h")).read()
    return re.findall(r"TFS_API\s+[\w\s\*]+?\b(tfs_\w+)\s*\(", h)


def test_header_declares_the_boundary():
    syms = declared_symbols()
    for s in ["tfs_create", "tfs_upload_data", "tfs_eval", "tfs_topk", "tfs_destroy", "tfs_last_error",
              "tfs_count_pixels", "tfs_default_opts", "tfs_bad_param_count", "tfs_set_profiling",
              "tfs_get_profile", "tfs_get_profile_kernels", "tfs_refine", "tfs_probe_l2_bandwidth", "tfs_eval_tf",
              "tfs_upload_timeseries", "tfs_weight_structure"]:
        assert s in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for s in declared_symbols():
        assert hasattr(lib, s), s


def test_defaults_and_create_fails_loudly_without_gpu(lib_path):
    from paper_2510_19047_b200 import api
    lib = api.load_library()
    o = api.tfs_opts()
    lib.tfs_default_opts(ctypes.byref(o))
    assert (o.half_width, o.adaptive_width, o.c_max, o.fresnel_mode) == (10, 1, 300.0, 0)
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(api.TfsError) as ei:      # no CPU fallback: creation must fail, loudly
            api.Tfs(64, 64, 5.0)
        assert ei.value.code in (api.TFS_ECUDA, api.TFS_ENOMEM)
    h = ctypes.c_void_p()
    assert lib.tfs_create(ctypes.byref(h), 0, 64, 5.0, 2, None) == api.TFS_EINVAL
    assert lib.tfs_create(ctypes.byref(h), 64, 64, 5.0, 4, None) == api.TFS_EINVAL      # 1, 2 or 3 channels
    assert lib.tfs_create(ctypes.byref(h), 64, 64, 5.0, 0, None) == api.TFS_EINVAL
    assert b"n_channels" in lib.tfs_last_error(None)
    assert lib.tfs_eval(None, None, 0, 1, None, None, None, None, None) == api.TFS_EINVAL


def test_product_does_not_import_oracle():
    # the product path (package + bench GPU arm) must never route through oracle/
    pkg = os.path.join(ROOT, "paper_2510_19047_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
