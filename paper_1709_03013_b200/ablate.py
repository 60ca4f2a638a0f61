"""Timing ablations of the fp4 tensor kernel (developer aid; profiles/r1f… and r1g… quote its output).

    python -m paper_1709_03013_b200.ablate --config 2 --debug 0,14,9,63,64

The script builds and loads libcsg_ablate.so -- the library's sources compiled with -DCSG_ABLATE, which adds the
ablation switches to the fp4 instantiation of tensor_action_kernel and exports csg_set_debug -- INSTEAD of libcsg.so
(the product library has neither).  For every value of --debug it calls csg_set_debug (bits: 1 no MMA issue, 2 no expansion arithmetic, 4 no
operand stores, 8 no bucketing in the epilogue, 16 no fence before publishing a stage, 32 no packed-bit ring, 64 free-running
producers, 128 no prefill before the epilogue, 256 no open-range masks; any non-zero value gives WRONG counts), and the
CUDA-event time of the interval kernel (csg_last_kernel_ms) of four calls is printed.  Needs a B200.

The run-time switches cost the -DCSG_ABLATE build 28 % against the product, so absolute numbers come from --static:

    python -m paper_1709_03013_b200.ablate --config 3 --static "" CSG_STATIC_DBG=8 CSG_STATIC_DBG=1 CSG_STATIC_DBG=64 \
        CSG_STATIC_DBG=128 CSG_PREFILL_GROUPS=3

builds one measurement library per item (libcsg_variant_<macros>.so: the product's sources with those -D macros, several
per item separated by commas; "" = the product's own settings) with the switch as a COMPILE-TIME constant, so that
whatever is left runs at product speed, loads each in turn and prints the same kernel times (table of
compile-time ablations).  CSG_STATIC_DBG takes the bits above (wrong counts); CSG_PREFILL_GROUPS, CSG_BITS_BUFS (at most 5: shared memory),
CSG_WHOLE_GROUP, CSG_SCALE_CLASSES, CSG_A_IN_TMEM are the kernel's tuning macros (right counts).
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def run_static(args):
    """One measurement library per --static item, each through plain ctypes (the binding holds ONE library)."""
    import ctypes
    import numpy as np
    import torch
    import csg_inputs
    from paper_1709_03013_b200 import _build
    cfg = csg_inputs.CONFIGS[args.config]
    N, dim, eps, kmax = cfg["N"], cfg["dim"], cfg["eps"], cfg["kmax"]
    _, bits = csg_inputs.make_config(cfg)
    d = torch.from_numpy(bits.view(np.int64)).cuda()
    counts = torch.empty(kmax + 1, dtype=torch.int64, device="cuda")
    S = torch.empty(1, dtype=torch.float64, device="cuda")
    vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    for item in args.static:
        defines = tuple(x for x in item.split(",") if x)
        path = _build.build(defines=defines) if defines else _build.build()
        lib = ctypes.CDLL(path)
        lib.csg_action.argtypes = [vp, i64, ci, dbl, ci, vp, vp, vp]
        lib.csg_set_sparse.argtypes = [ci]
        lib.csg_set_variant.argtypes = [ci]
        lib.csg_set_kernel_timing.argtypes = [ci]
        lib.csg_last_kernel_ms.argtypes = [ctypes.POINTER(ctypes.c_float)]
        lib.csg_set_variant(3)
        lib.csg_set_sparse(args.sparse)
        lib.csg_set_kernel_timing(1)
        ms = []
        for _ in range(args.runs + 2):
            rc = lib.csg_action(d.data_ptr(), N, dim, eps, kmax, counts.data_ptr(), S.data_ptr(), None)
            assert rc == 0, rc
            torch.cuda.synchronize()
            f = ctypes.c_float()
            lib.csg_last_kernel_ms(ctypes.byref(f))
            ms.append(f.value)
        print("%s sparse=%d static[%s] kernel ms %s  counts[0..3] %s" % (
            cfg["name"], args.sparse, item or "product", " ".join("%.3f" % m for m in ms[2:]), counts[:4].tolist()), flush=True)
        lib.csg_shutdown()


def main():
    import ctypes
    import torch
    import csg_inputs
    import paper_1709_03013_b200 as csg
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2, help="index into csg_inputs.CONFIGS")
    ap.add_argument("--debug", default="0,14,9,63,64", help="comma-separated CSG_DEBUG values")
    ap.add_argument("--runs", type=int, default=4)
    ap.add_argument("--sparse", type=int, default=0, help="csg_set_sparse mode: 0 auto, 1 on, 2 off (dense sweep)")
    ap.add_argument("--static", nargs="*", default=None,
                    help='compile-time measurement builds, one per item: "MACRO=V[,MACRO=V...]"; "" = the product settings')
    args = ap.parse_args()
    if args.static is not None:
        return run_static(args)
    csg.LIB_PATH = csg._build.build(ablate=True)       # never the product library
    lib = csg.load()
    lib.csg_set_debug.argtypes = [ctypes.c_int]
    cfg = csg_inputs.CONFIGS[args.config]
    N, dim = cfg["N"], cfg["dim"]
    _, bits = csg_inputs.make_config(cfg)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(args.sparse)
    csg.csg_set_kernel_timing(True)
    for dbg in [int(x) for x in args.debug.split(",")]:
        lib.csg_set_debug(dbg)
        ms = []
        for _ in range(args.runs):
            csg.csg_action(d, N, dim, 1.0, 3)
            torch.cuda.synchronize()
            ms.append(csg.csg_last_kernel_ms())
        print("%s sparse=%d CSG_DEBUG=%-4d kernel ms %s" % (cfg["name"], args.sparse, dbg, " ".join("%.3f" % m for m in ms)), flush=True)
    lib.csg_set_debug(0)
    csg.csg_set_kernel_timing(False)
    csg.csg_set_variant(csg.VARIANT_AUTO)


if __name__ == "__main__":
    main()
