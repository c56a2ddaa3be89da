"""CPU-side checks of the boundary: libnbk.so loads, exports every symbol include/nbk.h
declares, validates arguments, and fails loudly (no fallback) when there is no CUDA device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_0707_0438_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared():
    text = open(os.path.join(ROOT, "include", "nbk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nbk_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    names = _declared()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), f"{name} declared in nbk.h but not exported by libnbk.so"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and nbk.h disagree"


def test_binding_has_same_names():
    for name in binding.EXPORTS:
        if name in ("nbk_strerror", "nbk_last_cuda_error"):
            continue
        assert callable(getattr(binding, name)), f"binding lacks {name}"


def test_strerror_and_version(lib):
    assert lib.nbk_strerror(0) == b"ok"
    for code in range(-5, 0):
        assert len(lib.nbk_strerror(code)) > 3
    assert b"sm_100a" in lib.nbk_version()


def test_null_and_bad_arguments(lib):
    assert lib.nbk_open(None, 0, 16, 16, None) == binding.NBK_EINVAL
    ctx = ctypes.c_void_p()
    assert lib.nbk_open(ctypes.byref(ctx), 0, 0, 16, None) == binding.NBK_EINVAL
    assert lib.nbk_open(ctypes.byref(ctx), 0, 16, -1, None) == binding.NBK_EINVAL
    assert lib.nbk_open_ws(ctypes.byref(ctx), 0, 16, 16, None, None, 1024) == binding.NBK_EINVAL
    assert lib.nbk_workspace_bytes(0, 0, 16) == binding.NBK_EINVAL
    assert lib.nbk_calc_lasthalf_f64(None, 1, None, None, None) == binding.NBK_EINVAL
    assert lib.nbk_close(None) == binding.NBK_OK
    assert lib.nbk_npipes(None) == binding.NBK_EINVAL
    assert lib.nbk_set_ti(None, 0.0) == binding.NBK_EINVAL
    assert lib.nbk_sync(None) == binding.NBK_EINVAL
    assert lib.nbk_calc_firsthalf(None, 1, 1, None, None, None, 0.0, 0) == binding.NBK_EINVAL
    assert lib.nbk_calc_lasthalf(None, 1, None, None, None) == binding.NBK_EINVAL
    assert lib.nbk_hermite_evolve(None, 1, None, None, None, 0.0, 1.0, 0.01, 0.0625, None) == binding.NBK_EINVAL
    assert lib.nbk_hermite_evolve_dev(None, 1, None, None, None, 0.0, 1.0, 0.01, 0.0625, None) == binding.NBK_EINVAL
    assert lib.nbk_get_neighbours(None, 1, None, None) == binding.NBK_EINVAL
    assert lib.nbk_get_neighbours_dev(None, 1, None, None) == binding.NBK_EINVAL
    assert lib.nbk_calc_batch(None, 1, None, None, None, None, None, 0.0, 0, None, None) == binding.NBK_EINVAL
    assert lib.nbk_calc_batch_dev(None, 1, None, None, None, None, None, 0.0, 0, None, None) == binding.NBK_EINVAL


def test_no_gpu_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    ctx = ctypes.c_void_p()
    rc = lib.nbk_open(ctypes.byref(ctx), 0, 1024, 1024, None)
    assert rc in (binding.NBK_ECUDA, binding.NBK_ENOMEM) and not ctx.value
    with pytest.raises(binding.NbkError):
        binding.nbk_open(0, 1024, 1024)


def test_product_does_not_import_oracle():
    """The CUDA path neither imports, links, includes nor dlopens anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_0707_0438_b200")
    pat = re.compile(r"(^\s*(import|from)\s+oracle\b)|(import_module\(.oracle)|(#include\s*[\"<][^\">]*oracle)"
                     r"|(liboracle)|(oracle[/\\.](nbody_oracle|c_oracle|hermite_oracle))", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not pat.search(src), f"{f} reaches into the oracle"
