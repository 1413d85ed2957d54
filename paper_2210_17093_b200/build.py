"""Build step: compile the CUDA sources under csrc/ into shared libraries, in-tree, for sm_100a only.

  libqsgw_sigma.so             the product (include/qsgw_sigma.h)
  libqsgw_sigma_testhooks.so   the same sources with -DQSGW_SIGMA_TEST_HOOKS (adds qsgw_sigma_copy_workspace); tests only
  libqsgw_fp64_probe.so        csrc/probe/fp64_probe.cu, the FP64 issue-rate probe bench.py measures its roofline with
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libqsgw_sigma.so")
TESTHOOKS_LIB_PATH = os.path.join(_HERE, "libqsgw_sigma_testhooks.so")
PROBE_LIB_PATH = os.path.join(_HERE, "libqsgw_fp64_probe.so")
SOURCES = ["qsgw_sigma.cu"]
HEADERS = sorted(f for f in os.listdir(CSRC) if f.endswith(".cuh")) + [os.path.join("..", "..", "include", "qsgw_sigma.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--shared", "-Xcompiler", "-fPIC", "-cudart", "shared",
]


def _stale(out: str, deps) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(d) > t for d in list(deps) + [os.path.abspath(__file__)])


def _nvcc(out: str, sources, extra=(), verbose: bool = False) -> None:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = out + f".tmp{os.getpid()}"
    cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *sources]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)


def build_library(force: bool = False, verbose: bool = False, test_hooks: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a ... -> libqsgw_sigma.so (or the test-hooks variant)"""
    out = TESTHOOKS_LIB_PATH if test_hooks else LIB_PATH
    srcs = [os.path.join(CSRC, f) for f in SOURCES]
    if force or _stale(out, srcs + [os.path.join(CSRC, h) for h in HEADERS]):
        _nvcc(out, srcs, ["-DQSGW_SIGMA_TEST_HOOKS"] if test_hooks else [], verbose)
    return out


def build_probe(force: bool = False) -> str:
    src = os.path.join(CSRC, "probe", "fp64_probe.cu")
    if force or _stale(PROBE_LIB_PATH, [src]):
        _nvcc(PROBE_LIB_PATH, [src])
    return PROBE_LIB_PATH


def build_all(force: bool = False, verbose: bool = False):
    """All three libraries, compiled side by side."""
    with concurrent.futures.ThreadPoolExecutor(3) as ex:
        jobs = [ex.submit(build_library, force, verbose, False), ex.submit(build_library, force, False, True),
                ex.submit(build_probe, force)]
        return [j.result() for j in jobs]


if __name__ == "__main__":
    import sys
    for path in build_all(force="--force" in sys.argv, verbose="-v" in sys.argv):
        print(path)
