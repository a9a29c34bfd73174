"""The C-ABI library loads and exports every symbol include/hough.h declares (no compute calls, no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1311_2769_b200 import build
    return build.build()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "hough.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hough_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_four_named_calls():
    names = _declared_functions()
    for n in ("hough_plan_create", "hough_vote", "hough_find_peaks", "hough_assign_hits"):
        assert n in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared_functions():
        assert hasattr(lib, name), name
    from paper_1311_2769_b200 import EXPORTS
    assert sorted(EXPORTS) == _declared_functions()


def test_status_strings_and_version(lib_path):
    from paper_1311_2769_b200 import load_library, version
    lib = load_library()
    assert lib.hough_status_string(0) == b"ok"
    assert b"invalid" in lib.hough_status_string(-1)
    assert "sm_100a" in version()


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1311_2769_b200 import HoughPlan, HoughError
    with pytest.raises(HoughError):
        HoughPlan(256, 256, 1)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1311_2769_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower() or f == "__init__.py" and False, (dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1311_2769_b200" not in src and "from paper_1311_2769_b200" not in src
            assert "libhough_b200" not in src and "csrc" not in src


def test_static_fit_refuses_oversized_lists_before_any_cuda_call(lib_path):
    """hough_fit_circles_static keeps its scratch in a fixed array: a candidate capacity beyond
    HOUGH_FIT_STATIC_MAX_CANDIDATES must come back as HOUGH_ERR_TOO_LARGE (-5) with a message that names the limit, and
    plain argument errors as INVALID_ARG -- both decided on the host, so this runs without a GPU."""
    header = open(os.path.join(ROOT, "include", "hough.h")).read()
    limit = int(re.search(r"#define\s+HOUGH_FIT_STATIC_MAX_CANDIDATES\s+(\d+)", header).group(1))
    from paper_1311_2769_b200 import FIT_STATIC_MAX_CANDIDATES, load_library
    assert FIT_STATIC_MAX_CANDIDATES == limit
    lib = load_library()
    dummy = ctypes.create_string_buffer(64)                       # never dereferenced: the checks come first
    p = ctypes.cast(dummy, ctypes.c_void_p)
    rc = lib.hough_fit_circles_static(256, 3.8, None, 0, None, p, p, 1, limit + 1, None, p, p, None)
    assert rc == -5
    msg = lib.hough_status_string(rc)
    assert b"HOUGH_FIT_STATIC_MAX_CANDIDATES" in msg and b"no-allocation" in msg
    assert lib.hough_fit_circles_static(0, 3.8, None, 0, None, p, p, 1, 1, None, p, p, None) == -1      # n_phi <= 0
    assert lib.hough_fit_circles_static(256, 3.8, None, 0, None, p, None, 1, 1, None, p, p, None) == -1  # no offsets
    assert lib.hough_fit_circles_static(256, 3.8, None, 5, None, p, p, 1, 1, None, p, p, None) == -1     # hits without pointers
    assert lib.hough_fit_circles_static(256, 3.8, None, 0, None, p, p, 1, 0, None, None, None, None) == 0  # capacity 0: no-op
