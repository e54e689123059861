"""The C-ABI boundary without a GPU: the library builds, loads and exports every symbol that
include/monteray.h declares; the binding lists the same names; no compute call is made."""
import ctypes as C
import os
import re

import pytest

from paper_1706_07476_b200 import EXPORTS, LIB_PATH, load_library
from paper_1706_07476_b200 import build as mr_build


@pytest.fixture(scope="module")
def lib():
    mr_build.build()
    return load_library()


def declared_symbols(repo_root):
    text = open(os.path.join(repo_root, "include", "monteray.h")).read()
    return sorted(set(re.findall(r"MR_API\s+[\w\s\*]+?\b(mr_\w+)\s*\(", text)))


def test_header_symbols_exported(lib, repo_root):
    names = declared_symbols(repo_root)
    assert len(names) >= 15
    for nm in names:
        assert hasattr(lib, nm), f"{nm} declared in monteray.h but not exported by {LIB_PATH}"
    assert sorted(EXPORTS) == names, "binding.EXPORTS and monteray.h disagree"


def test_no_torch_types_in_header(repo_root):
    text = open(os.path.join(repo_root, "include", "monteray.h")).read()
    assert "at::" not in text and "c10::" not in text and "#include <torch" not in text


def test_create_argument_errors(lib):
    h = C.c_void_p()
    assert lib.mr_create(None, 0, 0) == 1  # MR_ERR_INVALID_ARG
    assert b"NULL" in lib.mr_last_error(None)
    assert lib.mr_create(C.byref(h), 0, 7) == 1
    assert h.value is None
    assert lib.mr_destroy(None) == 0


def test_create_fails_loudly_without_gpu(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    rc = lib.mr_create(C.byref(h), 0, 0)
    assert rc == 3, "without a CUDA device mr_create must return MR_ERR_CUDA (no CPU fallback)"
    assert h.value is None and len(lib.mr_last_error(None)) > 0


def test_product_does_not_import_oracle(repo_root):
    pkg = os.path.join(repo_root, "paper_1706_07476_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "vrc_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(repo_root, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(repo_root, "oracle", f)).read()
            assert "import paper_1706_07476_b200" not in text and "from paper_1706_07476_b200" not in text
            assert "monteray.h" not in text and "mr_device" not in text


def test_option_and_limit_constants_match_the_header(repo_root):
    """binding.py restates the MR_OPT_* / precision / location constants of monteray.h: keep them in step."""
    import paper_1706_07476_b200.binding as b

    text = open(os.path.join(repo_root, "include", "monteray.h")).read()
    found = dict(re.findall(r"\b(MR_(?:OPT|INFO|PRECISION|WHERE)_\w+)\s*=\s*(\d+)", text))
    assert len([k for k in found if k.startswith("MR_OPT_")]) >= 10
    paths = dict(re.findall(r"\b(MR_PATH_\w+)\s*=\s*(\d+)", text))
    assert sorted(int(v) for v in paths.values()) == sorted(b.MR_PATH_NAMES), "MR_PATH_* and binding.MR_PATH_NAMES differ"
    for name, value in found.items():
        assert hasattr(b, name), f"{name} is in monteray.h but not in binding.py"
        assert getattr(b, name) == int(value), name
    status = dict(re.findall(r"\b(MR_(?:OK|ERR_\w+))\s*=\s*(\d+)", text))
    for name, value in status.items():
        assert getattr(b, name) == int(value), name
