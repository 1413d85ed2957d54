"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/qsgw_sigma.h declares; argument validation that happens before any device work; and the
product never routes through the oracle."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(test_hooks=False):
    text = open(os.path.join(ROOT, "include", "qsgw_sigma.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    if not test_hooks:
        text = re.sub(r"#ifdef QSGW_SIGMA_TEST_HOOKS.*?#endif", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qsgw_[a-z0-9_]+)\s*\(", text)))


def _exported(path):
    out = subprocess.run(["nm", "-D", "--defined-only", path], check=True, capture_output=True, text=True).stdout
    return sorted(set(re.findall(r"\bT (qsgw_[a-z0-9_]+)$", out, flags=re.M)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2210_17093_b200 import build, binding
    path = build.build_library()
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert "qsgw_sigma_create" in declared and "qsgw_sigma_build" in declared and "qsgw_sigma_destroy" in declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/qsgw_sigma.h but not exported"
    assert _exported(path) == declared                  # ... and nothing else: no probe, no test hook in the product
    assert sorted(binding.EXPORTS) == declared          # the Python binding carries the same names
    import paper_2210_17093_b200 as pkg
    for name in declared:
        assert callable(getattr(pkg, name))
    assert pkg.qsgw_sigma_version() >= 100


def test_test_hook_and_probe_live_in_their_own_libraries():
    from paper_2210_17093_b200 import build
    hooks = _declared_symbols(test_hooks=True)
    assert "qsgw_sigma_copy_workspace" in hooks and "qsgw_sigma_copy_workspace" not in _declared_symbols()
    assert _exported(build.build_library(test_hooks=True)) == hooks
    assert _exported(build.build_probe()) == ["qsgw_fp64_probe"]


def test_create_rejects_bad_sizes_before_touching_the_device():
    import paper_2210_17093_b200 as pkg
    lib = pkg.load_library()
    h = ctypes.c_void_p()
    bad = [(1, 1, 4, 4, 0), (8, 0, 4, 4, 0), (8, 8, 4, 4, 0), (8, 2, 0, 4, 0), (8, 2, 4, 0, 0), (8, 2, 4, 4, -1)]
    for n_mo, n_occ, n_aux, n_pole, s_block in bad:
        rc = lib.qsgw_sigma_create(ctypes.byref(h), n_mo, n_occ, n_aux, n_pole, s_block, None)
        assert rc == pkg.QSGW_SIGMA_ERR_INVALID_ARG and not h.value
        assert b"create" in lib.qsgw_sigma_last_error(None)
    assert lib.qsgw_sigma_create(None, 8, 2, 4, 4, 0, None) == pkg.QSGW_SIGMA_ERR_INVALID_ARG
    assert lib.qsgw_sigma_destroy(None) == pkg.QSGW_SIGMA_OK


def test_no_cpu_fallback_without_a_device():
    import torch
    import paper_2210_17093_b200 as pkg
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less container")
    with pytest.raises(pkg.QsgwSigmaError) as ei:
        pkg.qsgw_sigma_create(24, 5, 80, 95)
    assert ei.value.code == pkg.QSGW_SIGMA_ERR_CUDA


def test_product_does_not_import_or_link_the_oracle():
    pkg_dir = os.path.join(ROOT, "paper_2210_17093_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2210_17093_b200" not in text and "from paper_2210_17093_b200" not in text
            assert "csrc" not in text or f.endswith(".c")   # the C file only names csrc/ in its header comment


def test_stats_struct_layout_matches_the_header():
    """The ctypes mirror of qsgw_sigma_stats must list the header's fields in the header's order with the header's types."""
    from paper_2210_17093_b200 import binding
    text = open(os.path.join(ROOT, "include", "qsgw_sigma.h")).read()
    body = re.search(r"typedef struct qsgw_sigma_stats \{(.*?)\} qsgw_sigma_stats;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    declared = [(t, n) for t, n in re.findall(r"\b(double|int64_t)\s+(\w+)\s*;", body)]
    mirror = [("double" if c is ctypes.c_double else "int64_t", n) for n, c in binding.qsgw_sigma_stats._fields_]
    assert declared == mirror
    assert ctypes.sizeof(binding.qsgw_sigma_stats) == 8 * len(declared)
