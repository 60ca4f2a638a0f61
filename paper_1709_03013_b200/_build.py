"""Build libcsg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcsg.so")
ABLATE_LIB_PATH = os.path.join(_HERE, "libcsg_ablate.so")    # -DCSG_ABLATE build, only ever loaded by ablate.py
_CSRC = os.path.join(_HERE, "csrc")
_INCLUDE = os.path.join(os.path.dirname(_HERE), "include")


def _sources():
    srcs = [os.path.join(_INCLUDE, "csg.h")]
    for name in sorted(os.listdir(_CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            srcs.append(os.path.join(_CSRC, name))
    return srcs


def needs_build(path=None):
    path = path or LIB_PATH
    if not os.path.exists(path):
        return True
    t = os.path.getmtime(path)
    return any(os.path.getmtime(s) > t for s in _sources())


def build(force=False, verbose=False, ablate=False, defines=()):
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -> paper_1709_03013_b200/libcsg.so
    ablate=True builds libcsg_ablate.so instead: the same sources with -DCSG_ABLATE, i.e. with the timing-ablation
    switches of the fp4 kernel and csg_set_debug compiled in (wrong counts when set; never the product library).
    defines: extra -D macros of a measurement build (ablate.py --static); such a build goes to
    libcsg_variant_<macros>.so, NEVER to libcsg.so."""
    out = ABLATE_LIB_PATH if ablate else LIB_PATH
    if defines:
        tag = "_".join(sorted(defines)).replace("=", "-")
        tag = "".join(ch if (ch.isalnum() or ch in "-_") else "_" for ch in tag)
        out = os.path.join(_HERE, "libcsg_variant_%s%s.so" % ("ablate_" if ablate else "", tag))
    if not force and not needs_build(out):
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [
        nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
        "-shared", "-Xcompiler", "-fPIC", "-o", out, os.path.join(_CSRC, "csg.cu"),
    ]
    if ablate:
        cmd.insert(1, "-DCSG_ABLATE")
    for d in defines:
        cmd.insert(1, "-D" + d)
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return out
