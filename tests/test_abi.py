"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/csg.h declares,
validates arguments, and fails loudly (no CPU fallback) when there is no CUDA device."""
import os
import re

import numpy as np
import pytest

import paper_1709_03013_b200 as csg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    if csg._build.needs_build():
        csg.build()
    return csg.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "csg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(csg_[a-z_0-9]+)\s*\(", text)))


def test_exports_match_header(lib):
    names = declared_functions()
    assert sorted(csg.EXPORTS) == names
    for n in names:
        assert getattr(lib, n) is not None


def test_no_environment_switches_in_the_product_library(lib):
    """The timing-ablation switches (wrong counts when set) live only in the -DCSG_ABLATE build: libcsg.so reads no
    environment variable and exports no csg_set_debug."""
    import subprocess
    syms = subprocess.run(["nm", "-D", csg.LIB_PATH], capture_output=True, text=True, check=True).stdout
    assert "csg_set_debug" not in syms               # (getenv itself is imported by the static CUDA runtime)
    blob = open(csg.LIB_PATH, "rb").read()
    assert b"CSG_DEBUG" not in blob and b"CSG_NO_THROTTLE" not in blob and b"CSG_" + b"ABLATE" not in blob
    for src in ("csg.cu", "tensor_kernel.cuh", "bitset_kernel.cuh", "link_kernel.cuh", "peak_kernels.cuh"):
        assert "getenv" not in open(os.path.join(ROOT, "paper_1709_03013_b200", "csrc", src)).read(), src


def test_throttle_setter(lib):
    for mode in (csg.THROTTLE_ON, csg.THROTTLE_OFF, csg.THROTTLE_AUTO):
        csg.csg_set_throttle(mode)
    with pytest.raises(csg.CsgError) as e:
        csg.csg_set_throttle(3)
    assert e.value.code == -9


def test_row_stride(lib):
    assert [csg.csg_row_stride_words(n) for n in (1, 255, 256, 257, 1024, 131072)] == [4, 4, 4, 8, 16, 2048]
    assert csg.csg_row_stride_words(0) == 0


def test_strerror_distinct(lib):
    texts = {csg.csg_strerror(c) for c in range(0, -13, -1)}
    assert len(texts) == 13 and "unknown" in csg.csg_strerror(-99)


def test_variant_setter(lib):
    csg.csg_set_variant(csg.VARIANT_BITSET)
    assert csg.csg_effective_variant(1 << 17) == csg.VARIANT_BITSET
    csg.csg_set_variant(csg.VARIANT_AUTO)
    assert csg.csg_effective_variant(1024) == csg.VARIANT_BITSET
    assert csg.csg_effective_variant(1025) == csg.VARIANT_TENSOR_FP4
    assert csg.csg_effective_variant(1 << 17) == csg.VARIANT_TENSOR_FP4
    with pytest.raises(csg.CsgError) as e:
        csg.csg_set_variant(7)
    assert e.value.code == -9


@pytest.mark.parametrize("kwargs,code", [
    (dict(N=0), -2), (dict(dim=3), -4), (dict(eps=0.0), -5), (dict(eps=1.5), -5), (dict(eps=float("nan")), -5),
    (dict(kmax=-1), -6), (dict(kmax=1), -6), (dict(dim=4, kmax=2), -6),
])
def test_argument_validation_precedes_cuda(lib, kwargs, code):
    args = dict(N=8, dim=2, eps=1.0, kmax=3)
    args.update(kwargs)
    bits = np.zeros((8, 4), np.uint64)
    with pytest.raises(csg.CsgError) as e:
        csg.csg_action_host(bits, args["N"], args["dim"], args["eps"], args["kmax"])
    assert e.value.code == code


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    bits = np.zeros((8, 4), np.uint64)
    with pytest.raises(csg.CsgError) as e:
        csg.csg_action_host(bits, 8, 2, 1.0, 3)
    assert e.value.code == -8


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1709_03013_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("no CPU fallback", ""), os.path.join(dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1709_03013_b200 import" not in open(os.path.join(ROOT, "oracle", f)).read()
