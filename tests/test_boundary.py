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
