"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol
include/fann.h declares.  No compute call is made here."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2409_16576_b200.build import build
    return build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "fann.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fann_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ("fann_load_codes", "fann_build_lut", "fann_dedup_scan_topk"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    names = declared_functions()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"{n} declared in fann.h but not exported"
    out = subprocess.check_output(["nm", "-D", "--defined-only", lib_path]).decode()
    exported = set(re.findall(r" T (fann_[a-z_]+)", out))
    assert set(names) <= exported


def test_binding_mirrors_the_header(lib_path):
    import paper_2409_16576_b200 as fann
    for n in declared_functions():
        assert hasattr(fann, n), f"python binding lacks {n}"
    assert fann.fann_version().endswith("sm_100a")


def test_sass_is_sm100a_only(lib_path):
    out = subprocess.check_output(["cuobjdump", "--list-elf", lib_path]).decode()
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_no_cpu_fallback_without_a_device(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2409_16576_b200 as fann
    with pytest.raises(fann.FannError) as e:
        fann.fann_create(0)
    assert e.value.code == -2 and "no CPU fallback" in str(e.value)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2409_16576_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower(), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2409_16576_b200 import" not in txt and "import paper_2409_16576_b200" not in txt
