"""CPU-only checks of the boundary: liboat.so builds for sm_100a, loads, exports every symbol that
include/oat.h declares, and its entry points fail loudly (no CPU fallback) when there is no GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1304_2017_b200 import binding, build, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols(headers=("oat.h", "oat_probe.h")):
    names = set()
    for h in headers:
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(oat_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert {"oat_geometry_create", "oat_project", "oat_backproject", "oat_adjoint_check"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/*.h but not exported by liboat.so"
    assert set(binding.EXPORTS) == set(names)
    # the product header holds the paper's problem statement only: no probes, no kernel selection
    product = declared_symbols(("oat.h",))
    assert not [n for n in product if "measure" in n or "variant" in n or "kernel_ms" in n]


def test_binding_has_the_same_names():
    for n in declared_symbols():
        assert hasattr(binding, n), f"binding lacks {n}"


def test_library_is_built_for_sm_100a():
    out = os.popen(f"cuobjdump -lelf {build.LIB} 2>/dev/null").read()
    assert "sm_100a" in out


def test_descriptor_validation_needs_no_gpu(lib):
    w = wl.small()
    d, keep = binding.make_desc(w)
    h = ctypes.c_void_p()
    assert lib.oat_geometry_create(None, 0, ctypes.byref(h)) == binding.OAT_ERR_INVALID
    d.spacing = -1.0
    assert lib.oat_geometry_create(ctypes.byref(d), 0, ctypes.byref(h)) == binding.OAT_ERR_INVALID
    assert "spacing" in binding.oat_last_error()
    d.spacing = 0.5
    d.kband = 64
    assert lib.oat_geometry_create(ctypes.byref(d), 0, ctypes.byref(h)) == binding.OAT_ERR_INVALID
    d.kband = 8
    keep[0, 0] = np.nan
    assert lib.oat_geometry_create(ctypes.byref(d), 0, ctypes.byref(h)) == binding.OAT_ERR_INVALID
    assert h.value is None


def test_null_handles(lib):
    assert lib.oat_num_voxels(None) == -1
    assert lib.oat_num_samples(None) == -1
    assert lib.oat_project(None, None, None, None) == binding.OAT_ERR_INVALID
    assert lib.oat_backproject(None, None, None, None) == binding.OAT_ERR_INVALID
    lib.oat_geometry_destroy(None)                       # no-op
    assert b"sm_100a" in lib.oat_version()


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.OatError) as ei:
        binding.oat_geometry_create(wl.small())
    assert ei.value.code == binding.OAT_ERR_CUDA
    assert "no CPU fallback" in str(ei.value)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1304_2017_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oat_oracle" not in src and "oat_ref_" not in src and "import oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "oat_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "oat_oracle.c")).read()
    assert "paper_1304_2017_b200" not in osrc.replace("paper_1304_2017_b200/csrc", "")
    assert "#include \"oat" not in osrc
