"""Build libtfs.so in-tree with nvcc for sm_100a (the only target).

    python -m paper_2510_19047_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtfs.so")
SOURCES = [os.path.join(CSRC, "tfs.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "tfs_kernels.cuh"), os.path.join(CSRC, "tfs_frontend.cuh"), os.path.join(CSRC, "tfs_wdm.cuh"),
                  os.path.join(os.path.dirname(HERE), "include", "tfs.h")]


def nvcc_cmd(extra=(), out=None):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    return [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
            "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
            "-DTFS_BUILD", *extra, "-o", out or LIB, *SOURCES, "-lcudart"]


def build_variant(out: str, defines=()) -> str:
    """Compile a variant of the library (e.g. -DTFS_BOUNDS_CHECK, the debug build whose gather traps on an
    out-of-range index) to `out`; select it with the TFS_LIB_PATH environment variable."""
    cmd = nvcc_cmd([f"-D{d}" for d in defines], out=out)
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return out


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if os.environ.get("TFS_LIB_PATH"):          # an explicitly chosen prebuilt library: nothing to do
        return os.environ["TFS_LIB_PATH"]
    if not force and up_to_date():
        return LIB
    extra = ["-Xptxas", "-v"] if verbose else []
    cmd = nvcc_cmd(extra)
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
