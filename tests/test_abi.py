"""CPU-side checks of the boundary: the shared library loads, exports every symbol that
include/tdma.h declares, validates its arguments, and fails loudly (no CPU fallback) when there is
no CUDA device.  No compute call is made here."""
import ctypes
import os
import re

import pytest
import torch

import paper_2509_03933_b200 as tdma

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "tdma.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tdma_[a-z0-9_]+)\s*\(", text)))


def test_header_functions_are_exported_and_bound():
    lib = tdma.load_library()
    names = declared_functions()
    assert "tdma_plan_create" in names and "tdma_solve" in names and "tdma_plan_destroy" in names
    for name in names:
        assert hasattr(lib, name), "libtdma.so does not export %s" % name
        assert hasattr(tdma, name), "python binding lacks %s" % name
    assert sorted(tdma.EXPORTED_SYMBOLS) == names


def test_options_struct_matches_header():
    text = open(os.path.join(ROOT, "include", "tdma.h")).read()
    body = re.search(r"typedef struct tdma_options \{(.*?)\} tdma_options;", text, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"int\s+([a-z_]+)(\[\d+\])?;", body)
    assert [f[0] for f in fields] == [f[0] for f in tdma.tdma_options._fields_]
    assert ctypes.sizeof(tdma.tdma_options) == 4 * len(tdma.tdma_options._fields_) == 4 * 22


def test_version():
    assert tdma.tdma_version() >= 10000


@pytest.mark.parametrize("args,frag", [
    ((0, 8, 8, 1, 0), "dimensions"),
    ((8, 8, 8, 0, 0), "P must be"),
    ((8, 9, 8, 2, 0), "not divisible"),
    ((8, 8, 8, 8, 0), ">= 2 rows"),
    ((8, 8, 8, 2, 9), "batch"),
    ((8, 8, 8, 2, -1), "batch"),
])
def test_plan_create_rejects_bad_arguments(args, frag):
    with pytest.raises(tdma.TdmaError) as ei:
        tdma.tdma_plan_create(*args)
    assert frag in str(ei.value)


def test_unknown_dtype_rejected():
    with pytest.raises(tdma.TdmaError) as ei:
        tdma.tdma_plan_create(8, 8, 8, 2, 0, 1)
    assert "TDMA_F64" in str(ei.value)
    # a failed tdma_plan_create returns NULL; its status travels through tdma_last_status()
    assert ei.value.status == tdma.TDMA_ERR_UNSUPPORTED == tdma.tdma_last_status()


def test_last_status_follows_the_last_error():
    with pytest.raises(tdma.TdmaError) as ei:
        tdma.tdma_plan_create(0, 8, 8, 1, 0)
    assert ei.value.status == tdma.TDMA_ERR_INVALID_ARG == tdma.tdma_last_status()
    assert tdma.load_library().tdma_plan_destroy(None) == tdma.tdma_last_status() < 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful without a GPU")
def test_no_cpu_fallback_without_gpu():
    with pytest.raises(tdma.TdmaError) as ei:
        tdma.tdma_plan_create(8, 8, 8, 2, 0)
    assert "no CPU fallback" in str(ei.value)


def test_null_plan_is_an_error_not_a_crash():
    lib = tdma.load_library()
    assert lib.tdma_plan_get(None, 0) < 0
    assert lib.tdma_plan_destroy(None) < 0
    assert lib.tdma_solve(None, None, None, None, None, None, None) < 0
    assert lib.tdma_plan_workspace_bytes(None) == 0


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2509_03933_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2509_03933_b200" not in src and "libtdma" not in src
