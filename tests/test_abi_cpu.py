"""The C-ABI library loads and exports every symbol include/smre.h declares (no compute calls)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1503_03492_b200 as smre

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_header_symbols():
    lib = smre.load_library()
    header = open(os.path.join(ROOT, "include", "smre.h")).read()
    declared = set(re.findall(r"\b(smre_[a-z_0-9]+)\s*\(", header))
    assert declared == set(smre.exported_symbols)
    for name in declared:
        assert getattr(lib, name) is not None
    raw = ctypes.CDLL(smre.lib_path())
    for name in declared:
        getattr(raw, name)


def test_sass_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", smre.lib_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_argument_validation_needs_no_device():
    s, c = np.array([1, 2], np.int32), np.array([3.8, 9.6], np.float32)
    for args in [(0, 8, 1, s, c, 0), (8, 8, 0, s, c, 0), (8, 8, 1, s, c, 7),
                 (8, 8, 1, np.array([1, 9], np.int32), c, 0),      # side > min(H, W)
                 (8, 8, 1, np.array([2, 2], np.int32), c, 0),      # duplicate
                 (8, 8, 1, s, np.array([3.8, -1.0], np.float32), 0)]:
        with pytest.raises(smre.SmreError) as e:
            smre.smre_create(*args)
        assert e.value.status == smre.smre.SMRE_EINVAL
    with pytest.raises(smre.SmreError) as e:
        smre.smre_create(64, 64, 1, np.array([33], np.int32), np.array([1.0], np.float32), 0)
    assert e.value.status == smre.smre.SMRE_EUNSUPPORTED
    assert "SMRE_MAX_SIDE" in smre.smre_last_error()


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(smre.SmreError) as e:
        smre.smre_create(8, 8, 1, np.array([1, 2], np.int32), np.array([3.8, 9.6], np.float32), 0)
    assert e.value.status == smre.smre.SMRE_ECUDA and "no CPU path" in str(e.value)


def test_product_never_touches_oracle():
    """The product path must not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1503_03492_b200")
    pat = re.compile(r"(import\s+oracle|from\s+oracle|oracle/|smre_oracle|#include\s+\".*oracle)")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                for line in open(os.path.join(dirpath, f)):
                    code = line.split("//")[0].split("#")[0] if not line.lstrip().startswith("#include") else line
                    assert not pat.search(code), (f, line)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1503_03492_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "paper_1503_03492_b200/csrc/", "").replace("never imports paper_1503_03492_b200", "")
